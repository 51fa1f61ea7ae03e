"""Regenerates tests/golden/newell_self_terms.txt.

    python tests/golden/make_self_terms.py [--check]

Self-demagnetizing factors of the configs' cells and bodies from Aharoni's closed form for a uniformly magnetized
rectangular prism (J. Appl. Phys. 83, 3432 (1998), Eq. (1)), evaluated with mpmath at 50 significant digits and
printed to 12.  It imports nothing from oracle/ or from the product: the stored digits are independent of both.
--check compares with the committed file instead of writing it.
"""
import os
import sys

import mpmath as mp

mp.mp.dps = 50
HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "newell_self_terms.txt")

ROWS = [  # (Lx, Ly, Lz) in nm, tag
    ("# SURVEY.md §8(c) P3: self-terms of the configs' cells (Nyy = Nxx for these square cross-sections)", None),
    ((5, 5, 3), "P3"), ((2, 2, 1), "P3"),
    ("# SURVEY.md §8(c) P7: body factors N_self(Lx, Ly, Lz) of the configs", None),
    ((160, 160, 3), "P7-C1"), ((1024, 1024, 4), "P7-C2"), ((2048, 2048, 1), "P7-C3"), ((1024, 1024, 32), "P7-C5"),
]


def aharoni_Dz(A, B, C):
    """Demagnetizing factor along z of an A x B x C prism; a, b, c are the half-sides."""
    a, b, c = mp.mpf(A) / 2, mp.mpf(B) / 2, mp.mpf(C) / 2
    r = mp.sqrt(a * a + b * b + c * c)
    rab, rbc, rac = mp.sqrt(a * a + b * b), mp.sqrt(b * b + c * c), mp.sqrt(a * a + c * c)
    t = (b * b - c * c) / (2 * b * c) * mp.log((r - a) / (r + a))
    t += (a * a - c * c) / (2 * a * c) * mp.log((r - b) / (r + b))
    t += b / (2 * c) * mp.log((rab + a) / (rab - a))
    t += a / (2 * c) * mp.log((rab + b) / (rab - b))
    t += c / (2 * a) * mp.log((rbc - b) / (rbc + b))
    t += c / (2 * b) * mp.log((rac - a) / (rac + a))
    t += 2 * mp.atan(a * b / (c * r))
    t += (a ** 3 + b ** 3 - 2 * c ** 3) / (3 * a * b * c)
    t += (a * a + b * b - 2 * c * c) / (3 * a * b * c) * r
    t += c / (a * b) * (rac + rbc)
    t -= (rab ** 3 + rbc ** 3 + rac ** 3) / (3 * a * b * c)
    return t / mp.pi


def lines():
    out = ["# Lx Ly Lz (nm)   Nxx             Nzz              source"]
    for row, tag in ROWS:
        if tag is None:
            out.append(row)
            continue
        Lx, Ly, Lz = row
        nxx, nzz = aharoni_Dz(Ly, Lz, Lx), aharoni_Dz(Lx, Ly, Lz)
        out.append(f"{Lx} {Ly} {Lz}".ljust(17) + " " + mp.nstr(nxx, 12).ljust(15) + " " + mp.nstr(nzz, 12).ljust(16) + " " + tag)
    return out


if __name__ == "__main__":
    new = lines()
    if "--check" in sys.argv:
        old = [l.split() for l in open(OUT).read().splitlines() if l.strip()]
        ok = all(a.split() == b for a, b in zip(new, old)) and len(new) == len(old)
        print("golden file matches" if ok else "golden file DIFFERS")
        sys.exit(0 if ok else 1)
    open(OUT, "w").write("\n".join(new) + "\n")
    print(f"wrote {OUT}")
