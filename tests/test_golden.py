"""The oracle against the stored closed-form values of tests/golden/ (written by tests/golden/make_golden.py from the
paper's formulas in 50-digit arithmetic, without the oracle): eq. 9 / 15 / 16 and the
axis-aligned box of north_star / pin P1."""
import os

import numpy as np

import oracle
from workloads.meshes import box_mesh

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_g_matches_stored_eq9_eq15_eq16():
    rows = _rows("g_closed_forms.txt")
    assert {r[0] for r in rows} == {"eq9", "eq15", "eq16"}
    for kind, a, b, c, re, im in rows:
        got = oracle.g_fun(float(a), float(b), float(c))
        want = complex(float(re), float(im))
        # the arguments are stored as decimal strings; the oracle sees their double roundings: |dg| <= ~1e-16 * |args|
        assert abs(got - want) <= 2e-14, (kind, a, b, c, got, want)


def test_box_spectrum_matches_stored_closed_form():
    rows = _rows("box_spectrum.txt")
    v, f = box_mesh((0.0625, -0.125, 0.03125), (0.25, 0.1875, 0.3125))   # exactly representable in fp32
    k = 2.0 * np.pi * np.array([[float(r[0]), float(r[1]), float(r[2])] for r in rows])
    for mode, col in ((0, 3), (1, 5)):
        got = oracle.mesh_ft_forward(v, f, k, mode)
        want = np.array([complex(float(r[col]), float(r[col + 1])) for r in rows])
        assert np.abs(got - want).max() <= 1e-13, (mode, np.abs(got - want).max())
