"""Re-derive tests/golden/lattice_constants.txt from shell multiplicities.

Independent of oracle/ and of the CUDA path: only `math`.  r_3(k) = number of
(a,b,c) in Z^3 with a^2+b^2+c^2 = k: 6,12,8,6,24,24,0,12,30 for k = 1..9;
r_2(k): 4,4,0,4,8,0,0,4,4.  w = re/r - 1 (Eq.3), n0 = sum w
(Eq.5 on the lattice), lambda = sum r^2 w / sum w.
"""
import math
import os

R3 = {1: 6, 2: 12, 3: 8, 4: 6, 5: 24, 6: 24, 7: 0, 8: 12, 9: 30}
R2 = {1: 4, 2: 4, 3: 0, 4: 4, 5: 8, 6: 0, 7: 0, 8: 4, 9: 4}


def consts(mult, re, w=None):
    if w is None:
        w = lambda r: re / r - 1.0                      # PAPER.md:123 Eq.3
    sw = sum(m * w(math.sqrt(k)) for k, m in mult.items() if k < re * re)
    sr = sum(m * k * w(math.sqrt(k)) for k, m in mult.items() if k < re * re)
    cnt = sum(m for k, m in mult.items() if k < re * re)
    return sw, sr / sw, cnt


def main():
    rows = []
    for tag, mult in (("3d", R3), ("2d", R2)):
        for re in (2.1, 3.1):
            n0, lam, cnt = consts(mult, re)
            rows.append((f"n0_{tag}_{re}", n0, "P:134 Eq.5 + P:123 Eq.3 on the cubic lattice"))
            rows.append((f"lambda_{tag}_{re}", lam, "P:174, in units of l0^2"))
            rows.append((f"count_{tag}_{re}", cnt, "number of lattice neighbours"))
    for tag, mult in (("3d", R3), ("2d", R2)):
        for re in (2.1, 3.1):
            n0, lam, cnt = consts(mult, re, lambda r: (1.0 - r / re) ** 3)   # PAPER.md:128 Eq.4
            rows.append((f"n0_eq4_{tag}_{re}", n0, "P:134 Eq.5 + P:128 Eq.4 on the cubic lattice"))
            rows.append((f"lambda_eq4_{tag}_{re}", lam, "P:174 with the Eq.4 kernel, in units of l0^2"))
    n0 = consts(R3, 2.1)[0]
    w = lambda k: 2.1 / math.sqrt(k) - 1.0
    rows.append(("n_depth1_3d_2.1", n0 - w(4), "misses one (2,0,0) neighbour (T3)"))
    rows.append(("n_face_3d_2.1", n0 - (w(1) + 4 * w(2) + 4 * w(3) + w(4)),
                 "face particle misses 1+4+4+1 neighbours of shells 1,2,3,4 (T3)"))
    rows.append(("eos_1.01", 1000.0 * 100.0 / 7.0 * (1.01 ** 7 - 1.0),
                 "P:150 Eq.7 with rho=1000 c0=10 gamma=7 n*/n0=1.01 (T7)"))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "lattice_constants.txt")
    with open(out, "w") as f:
        for k, v, c in rows:
            f.write(f"{k} {v!r}  # {c}\n")


if __name__ == "__main__":
    main()
