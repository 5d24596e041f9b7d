"""Writes the text fixtures of tests/golden/ from closed forms only (50-digit mpmath); it imports neither the oracle
nor the CUDA path, so the stored values are fixed by the paper's formulas and the mathematics alone.

    python tests/golden/make_golden.py

  g_closed_forms.txt   eq. 9 (reading R1), eq. 15, eq. 16 at fixed arguments
  box_spectrum.txt     volume- and surface-mode FT of an axis-aligned box (north_star's cube pin; SURVEY.md pin P1):
                       volume  F = e^{-ik.c} prod_a S_a,  S_a = 2 sin(k_a h_a)/k_a (-> 2 h_a at k_a = 0)
                       surface F = e^{-ik.c} [2cos(k_x h_x) S_y S_z + 2cos(k_y h_y) S_x S_z + 2cos(k_z h_z) S_x S_y]
"""
import os

import mpmath as mp

mp.mp.dps = 50
HERE = os.path.dirname(os.path.abspath(__file__))


def eq9(a, b, c):
    E = lambda x: mp.e ** (-1j * x)
    return -E(a) / ((a - b) * (a - c)) - E(b) / ((b - c) * (b - a)) - E(c) / ((c - a) * (c - b))


def eq15(t, u):
    E = lambda x: mp.e ** (-1j * x)
    return 1j * E(t) / (t - u) + E(t) / (t - u) ** 2 - E(u) / (t - u) ** 2


def eq16(u):
    return mp.e ** (-1j * u) / 2


def fmt(z):
    return f"{mp.nstr(mp.re(z), 20)} {mp.nstr(mp.im(z), 20)}"


def write_g():
    rows = ["# kind a b c Re(g) Im(g)   -- eq9: PAPER.md:162; eq15 (a=b): PAPER.md:203; eq16 (a=b=c): PAPER.md:208"]
    for a, b, c in [(0.3, 1.7, -2.2), (10.5, -3.25, 4.0), (100.0, 101.5, 97.0), (-0.001, 0.002, 0.004), (5.0, 5.5, 40.0)]:
        rows.append(f"eq9 {a} {b} {c} {fmt(eq9(mp.mpf(a), mp.mpf(b), mp.mpf(c)))}")
    for t, u in [(0.7, 2.9), (-3.0, 3.0), (50.0, 50.25), (1.0, 200.0)]:
        rows.append(f"eq15 {t} {t} {u} {fmt(eq15(mp.mpf(t), mp.mpf(u)))}")
    for u in [0.0, 1.25, -77.0]:
        rows.append(f"eq16 {u} {u} {u} {fmt(eq16(mp.mpf(u)))}")
    open(os.path.join(HERE, "g_closed_forms.txt"), "w").write("\n".join(rows) + "\n")


def write_box():
    c = [mp.mpf("0.0625"), mp.mpf("-0.125"), mp.mpf("0.03125")]
    h = [mp.mpf("0.25"), mp.mpf("0.1875"), mp.mpf("0.3125")]
    rows = ["# box centre 0.0625 -0.125 0.03125, half-widths 0.25 0.1875 0.3125, box length L = 1 (k = 2 pi n)",
            "# n_x n_y n_z Re(F_vol) Im(F_vol) Re(F_surf) Im(F_surf)   -- closed forms of SURVEY.md pin P1"]
    for n in [(0, 0, 0), (1, 0, 0), (0, 2, 0), (0, 0, 3), (1, 1, 0), (1, -2, 3), (-5, 4, 7), (16, -16, 16), (3, 0, 11), (-9, -7, 2)]:
        k = [2 * mp.pi * x for x in n]
        S = [2 * mp.sin(k[a] * h[a]) / k[a] if n[a] != 0 else 2 * h[a] for a in range(3)]
        C = [2 * mp.cos(k[a] * h[a]) for a in range(3)]
        ph = mp.e ** (-1j * sum(k[a] * c[a] for a in range(3)))
        vol = ph * S[0] * S[1] * S[2]
        surf = ph * (C[0] * S[1] * S[2] + C[1] * S[0] * S[2] + C[2] * S[0] * S[1])
        rows.append(f"{n[0]} {n[1]} {n[2]} {fmt(vol)} {fmt(surf)}")
    open(os.path.join(HERE, "box_spectrum.txt"), "w").write("\n".join(rows) + "\n")


if __name__ == "__main__":
    write_g()
    write_box()
