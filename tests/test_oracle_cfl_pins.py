"""Pins of the oracle's maximum-CFL routine (paper's Listing 1) against what
the listing and arithmetic fix: the printed floor, closed forms for uniform flow, single-value spikes that
pin which metric, which neighbour and which periodic wrap each term uses, and the absolute value of the SUM."""
import os

import numpy as np

from oracle import ref

HERE = os.path.dirname(os.path.abspath(__file__))


def golden(key):
    for ln in open(os.path.join(HERE, "golden", "paper_values.txt")):
        if ln.strip().startswith(key):
            return float(ln.split("=")[1].split("#")[0])
    raise KeyError(key)


XC = np.array([0.0, 0.1, 0.4, 0.45, 1.0])       # nx = 4, dx = 0.1, 0.3, 0.05, 0.55
NX, NY, NZ, LY, LZ = 4, 6, 8, 3.0, 2.0          # dy = 0.5, dz = 0.25
DX = np.diff(XC)


def zeros():
    return np.zeros((NX + 1, NY, NZ)), np.zeros((NX, NY, NZ)), np.zeros((NX, NY, NZ))


def test_floor_is_the_papers_constant():
    u, v, w = zeros()
    assert ref.max_cfl(XC, LY, LZ, u, v, w) == golden("cfl_floor") == 1e-8


def test_uniform_flow_closed_form():
    u, v, w = zeros()
    u += 0.7; v -= 1.3; w += 2.1
    want = golden("cfl_half_factor") * (2 * 2.1 / 0.25 + 2 * 1.3 / 0.5 + 2 * 0.7 / DX.min())
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - want) <= 1e-14 * want


def test_single_u_spike_uses_the_widths_of_both_neighbour_cells():
    for face in (1, 2, 3):
        u, v, w = zeros()
        u[face, 2, 3] = -4.0
        want = 0.5 * 4.0 / min(DX[face - 1], DX[face])
        assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - want) <= 1e-14 * want
    u, v, w = zeros()
    u[0, 1, 1] = 4.0                              # wall face: only cell 0 sees it
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - 0.5 * 4.0 / DX[0]) <= 1e-13


def test_single_v_and_w_spikes_and_periodic_wrap():
    u, v, w = zeros()
    v[1, 0, 5] = 3.0                              # seen by cells j = 0 and j = ny-1 (wrap)
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - 0.5 * 3.0 / 0.5) <= 1e-14
    u, v, w = zeros()
    w[2, 4, 0] = -5.0                             # seen by cells k = 0 and k = nz-1 (wrap)
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - 0.5 * 5.0 / 0.25) <= 1e-14


def test_terms_take_the_absolute_value_of_the_sum_and_add_up():
    u, v, w = zeros()
    w[1, 1, 7] = 2.0; w[1, 1, 0] = -2.0           # wrap pair cancels in cell k = 7; cells k = 6 and k = 0 see one each
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - 0.5 * 2.0 / 0.25) <= 1e-14
    u, v, w = zeros()
    u[2, 3, 4] = 1.0; v[2, 3, 4] = 1.0; w[2, 3, 4] = 1.0      # all three terms meet in cell (2,3,4)
    want = 0.5 * (1.0 / 0.25 + 1.0 / 0.5 + 1.0 / DX[2])
    assert abs(ref.max_cfl(XC, LY, LZ, u, v, w) - want) <= 1e-14 * want


def test_scaling_and_sign_invariance():
    rng = np.random.default_rng(5)
    u = rng.standard_normal((NX + 1, NY, NZ)); v = rng.standard_normal((NX, NY, NZ)); w = rng.standard_normal((NX, NY, NZ))
    c = ref.max_cfl(XC, LY, LZ, u, v, w)
    assert abs(ref.max_cfl(XC, LY, LZ, -3 * u, -3 * v, -3 * w) - 3 * c) <= 1e-13 * c
    # halving every length doubles it
    assert abs(ref.max_cfl(XC / 2, LY / 2, LZ / 2, u, v, w) - 2 * c) <= 1e-13 * c
