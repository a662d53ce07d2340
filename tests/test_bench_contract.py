"""bench.py host logic (no GPU): the reference arm runs the CPU oracle and prints the contract's JSON line; the byte
model reproduces SURVEY 8(d)'s per-step figures."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "64sq",
                        "--steps", "3", "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "steps/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"]


def test_byte_model_matches_survey_8d():
    sys.path.insert(0, ROOT)
    import bench
    # 1024^2 p=2 fp64 226.8 MB; 256^3 p=2 fp64 5.269 GB; 2048^2 p=4 fp64 1.511 GB (fp32: 755.5 MB)
    for n, p, w, expect in (((1024, 1024), 2, 8, 226.8e6), ((256, 256, 256), 2, 8, 5.269e9), ((2048, 2048), 4, 8, 1.511e9),
                            ((2048, 2048), 4, 4, 755.5e6)):
        survey, design = bench.bytes_model(n, p, w)
        assert abs(sum(survey.values()) - expect) / expect < 1e-3
        assert sum(design.values()) < sum(survey.values())          # cross-step fusion moves fewer bytes than the per-pass ideal
        assert set(survey) == set(design)


def test_gpus_flag_spawns_ranks_itself():
    # `python bench.py --gpus 2` (no torchrun around it) must start two ranks; in the reference arm rank 0 alone works and
    # prints, rank 1 exits 0 -> exactly one JSON line with n_gpus = 2
    env = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        env.pop(k, None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--workload", "64sq",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2


def test_lib_override_is_refused():
    env = dict(os.environ, PF_LIBPF="/nonexistent/libpf_nocomp.so")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2"], capture_output=True, text=True,
                       timeout=600, env=env)
    assert r.returncode != 0 and "PF_LIBPF" in r.stderr


def test_design_byte_model_counts_the_carried_spectrum():
    # With c^ carried between steps (Algorithm 1) the last-axis kernel reads g^ and the carried c^, writes
    # the carried c^ and the z-form of c, and reads + writes every eta: (4 + 2p) arrays
    sys.path.insert(0, ROOT)
    import bench
    _, d2 = bench.bytes_model((1024, 1024), 2, 8)
    R = 1024 * 1024 * 8
    assert d2["col_y_fft_update_ifft"] == (4 + 2 * 2) * R == 67108864
    assert d2["row_c2r_nonlinear_r2c"] == 2 * 3 * R
    _, d3 = bench.bytes_model((256, 256, 256), 2, 8)
    Sp = 144 * 256 * 256 * 16                       # padded half spectrum: P2 = 144 complex per row
    assert d3["col_z_fft_update_ifft"] == (4 + 2 * 2) * Sp
    assert d3["col_y_fwd"] == 3 * (256 ** 3 * 8 + Sp) == d3["col_y_inv"]


def test_ab_switches_are_refused_and_recorded():
    sys.path.insert(0, ROOT)
    import bench
    env = dict(os.environ, PF_COL2D_LEGACY="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2"], capture_output=True, text=True,
                       timeout=600, env=env)
    assert r.returncode != 0 and "PF_COL2D_LEGACY" in r.stderr
    # every getenv("PF_...") of the host library that selects a code path is on bench.py's list
    import re
    src = open(os.path.join(ROOT, "paper_2306_04322_b200", "csrc", "pf.cu")).read()
    in_lib = set(re.findall(r'getenv\("(PF_[A-Z0-9_]+)"\)', src)) - {"PF_TRACE_FILE"}
    assert in_lib <= set(bench.SWITCHES), in_lib - set(bench.SWITCHES)


def test_ncu_traffic_is_quoted_only_for_the_sources_it_was_captured_from(tmp_path):
    sys.path.insert(0, ROOT)
    from paper_2306_04322_b200 import ncu_traffic as nt
    csvf = tmp_path / "cap.csv"
    csvf.write_text('"ID","Kernel Name","dram__bytes_read.sum","dram__bytes_write.sum"\n"","","Mbyte","Kbyte"\n'
                    '"0","void row_kernel<double, 512, 8, 1, 80, 3>(RowParams<T1>)","10.5","500"\n'
                    '"1","void row_kernel<double, 512, 8, 0, 80, 0>(RowParams<T1>)","99","0"\n'
                    '"2","void col2d_kernel<double, 1024, 8, 2>(Col2dParams<T1>)","20","1,000"\n'
                    '"3","void col2d_kernel<double, 1024, 8, 2>(Col2dParams<T1>)","22","1,000"\n'
                    '"4","void col_kernel<double, 256, 8, 4, 3>(ColParams<T1>)","1","0"\n')
    out = tmp_path / "t.json"
    nt.update("w", str(csvf), "ncu ...", str(out))
    doc = json.loads(out.read_text())["traffic"]["w"]
    assert doc["row_c2r_nonlinear_r2c"]["dram_bytes_per_launch"] == 11.0e6 and doc["row_c2r_nonlinear_r2c"]["launches"] == 1
    assert doc["col_y_fft_update_ifft"]["dram_bytes_per_launch"] == 22.0e6 and doc["col_y_fft_update_ifft"]["launches"] == 2
    assert doc["col_z_fft_update_ifft"]["source_hash"] == nt.source_hash("col_z_fft_update_ifft")
    # every header a kernel file includes is part of its hash
    import re
    for k, files in nt.KERNEL_SOURCES.items():
        seen, todo = set(), [files[0]]
        while todo:
            f = todo.pop()
            if f in seen:
                continue
            seen.add(f)
            todo += re.findall(r'#include "([a-z_0-9]+\.cuh)"', open(os.path.join(ROOT, "paper_2306_04322_b200", "csrc", f)).read())
        assert seen == set(files), (k, seen)
    # the committed file: bench.py quotes an entry only when its hash matches the tree
    import bench
    committed = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))["traffic"]
    for wl, ks in committed.items():
        for k, e in ks.items():
            val, _ = bench.ncu_traffic(wl, k)
            assert (val is not None) == (e["source_hash"] == nt.source_hash(k))
