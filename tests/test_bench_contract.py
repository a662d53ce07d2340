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
