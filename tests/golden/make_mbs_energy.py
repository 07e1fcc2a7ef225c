"""Writes tests/golden/mbs_energy.txt: draws of E_k / k_BT (Eq. 7; sampler reading U6 of DESIGN.md) from
the CPU oracle, as hexadecimal floats. Calls only oracle/. Run from the repo root: python tests/golden/make_mbs_energy.py"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", ".."))
from oracle.binding import Oracle  # noqa: E402

SEED = 0x0BADC0DE12345678


def main():
    o = Oracle((4, 4, 4), (4, 4, 4), 10, SEED)
    out = ["# E_k / k_BT ~ Gamma(3 (N_c - 1) / 2) of cell cid at step t (PAPER.md:64 Eq. (7); DESIGN.md reading U6), from oracle/ only",
           "# columns: cid t N_c value (C99 hexadecimal float); first row: the Philox seed",
           f"seed {SEED:#x}"]
    for Nc in (2, 3, 4, 7, 10, 11, 20, 33, 100):
        for cid, t in ((0, 0), (1, 0), (63, 5), (17, 1000), (42, 77777)):
            out.append(f"{cid} {t} {Nc} {float(o.mbs_energy(cid, t, Nc)).hex()}")
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "mbs_energy.txt"), "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
