"""Prints the distributed-shared-memory read rates of the current GPU (pf_dsmem_read_rate) as a markdown table.

    python -m paper_2306_04322_b200.dsmem_probe        # -> profiles/r3_dsmem.md
"""
from . import pf


def main():
    print("| cluster size | own shared memory, B/clk/SM | other CTAs' shared memory (DSMEM), B/clk/SM | ratio |")
    print("|---|---|---|---|")
    for cs in (1, 2, 4, 8, 16):
        try:
            own = pf.dsmem_read_rate(cs, False)
            rem = pf.dsmem_read_rate(cs, True) if cs > 1 else float("nan")
            print(f"| {cs} | {own:.1f} | {rem:.1f} | {rem / own:.2f} |")
        except pf.PfError as e:
            print(f"| {cs} | unavailable ({e}) | | |")


if __name__ == "__main__":
    main()
