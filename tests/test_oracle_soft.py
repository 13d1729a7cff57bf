"""Pins for the oracle's SOFT-STE mode (oracle/ovcs_soft.inc; BASELINE config 5) against what the paper and the
mathematics fix: its printed constants (tests/golden/soft_constants.txt), closed forms and limits of eq. (6), (8),
(9), (10), and Theorem 1/3 (soft forward == hard forward, tolerance 0) on the seeded synthetic cartridges."""
import ctypes as C
import math
import os

import numpy as np
import pytest

from oracle.ovcs_py import OracleVCS, lib
from vcs_inputs import make_workload

GOLD = {}
for line in open(os.path.join(os.path.dirname(__file__), "golden", "soft_constants.txt")):
    if line.strip() and not line.startswith("#"):
        name, val, tol = line.split()[:3]
        GOLD[name] = (float(val), float(tol))


def near(x, key):
    v, tol = GOLD[key]
    assert abs(x - v) <= tol, f"{key}: {x} vs paper {v} +- {tol}"


def relaxed(r, a, T, K=None):
    r = np.ascontiguousarray(r, dtype=np.float64)
    K = int(math.ceil(17 * T)) if K is None else K
    return lib().ovcs_soft_peek_relaxed(r.ctypes.data, len(r), a, T, K)


def test_peek_is_indexing():
    rng = np.random.default_rng(1)
    r = rng.integers(0, 256, 300).astype(np.float64)
    for a in (0, 1, 137, 299):
        assert lib().ovcs_soft_peek(r.ctypes.data, len(r), a) == r[a]          # eq. (1)/(6): forward value is r_a exactly


def test_relaxed_read_closed_forms():
    # constant tensor -> the constant (weights are normalised), at any T and at the clipped edges
    for T in (0.1, 1.0, 10.0):
        for a in (0, 3, 64, 127):
            assert abs(relaxed(np.full(128, 77.0), a, T) - 77.0) < 1e-9
    # T -> 0 collapses to indexing (L298)
    rng = np.random.default_rng(2); r = rng.integers(0, 256, 128).astype(np.float64)
    for a in (0, 50, 127):
        assert abs(relaxed(r, a, 0.02, K=4) - r[a]) < 1e-12
    # a single spike at distance d from the address contributes w_d = e^{-d/T} / sum_j e^{-|j|/T}
    T = 1.0; M = 4096; a = 2000; K = 17
    den = sum(math.exp(-abs(j) / T) for j in range(-K, K + 1))
    for d in (0, 1, -3, 9):
        r = np.zeros(M); r[a + d] = 255.0
        assert abs(relaxed(r, a, T) - 255.0 * math.exp(-abs(d) / T) / den) < 1e-9
    # symmetric in k: mirrored tensors give the same value
    r = rng.integers(0, 256, 101).astype(np.float64)
    assert abs(relaxed(r, 50, 3.0) - relaxed(r[::-1].copy(), 50, 3.0)) < 1e-9
    # geometric closed form of w_0 away from the edges: (1 - q) / (1 + q - 2 q^(K+1)), q = e^{-1/T}
    q = math.exp(-1 / T); w0 = (1 - q) / (1 + q - 2 * q ** (K + 1))
    r = np.zeros(M); r[a] = 1.0
    assert abs(relaxed(r, a, T) - w0) < 1e-12


def test_paper_constants_for_reads():
    # worst-case pull 255 (1 - w_0): addressed byte 0, every neighbour 255 (L459)
    T = 0.14
    r = np.full(4096, 255.0); r[2000] = 0.0
    pull = relaxed(r, 2000, T, K=40)
    near(pull, "pull_T014")
    near(510 * math.exp(-1 / T), "pull_bound_form_T014")
    assert pull < 0.5                                                         # so T = 0.14 still rounds to the hard byte
    near(1 / math.log(4 * 255), "T_max")
    # one max-amplitude neighbour at T = 0.20 (L437)
    r = np.zeros(4096); r[2001] = 255.0
    near(relaxed(r, 2000, 0.20, K=40), "neighbour_pull_T020")
    assert relaxed(r, 2000, 0.20, K=40) > 0.5


def test_gate_and_branch_margin():
    g = lib().ovcs_soft_gate
    for alpha in (2.0, 6.0, 20.0):
        assert abs(g(alpha, +1, 1.0) + g(alpha, +1, 0.0) - 1.0) < 1e-12       # sigma(x) + sigma(-x) = 1
        assert g(alpha, +1, 1.0) == g(alpha, -1, 0.0)                         # z = s(2f - 1)
        assert abs(g(alpha, +1, 1.0) - 1 / (1 + math.exp(-alpha))) < 1e-15
    assert g(60.0, +1, 1.0) == 1.0 and g(60.0, +1, 0.0) < 1e-20               # alpha -> inf: the hard branch
    # the rounded soft PC stays on the hard target iff |delta| < tau_b(alpha) = (1 + e^alpha) / 2 (L429)
    near(0.5 * (1 + math.exp(6.0)), "tau_b_alpha6")
    near(math.log(2 * 127 - 1), "alpha_min")
    for alpha in (3.0, 6.0):
        tau = 0.5 * (1 + math.exp(alpha))
        for delta in range(-128, 128):
            taken_soft = round(1000 + g(alpha, +1, 1.0) * delta)               # flag set, branch-when-set: hard target 1000 + delta
            assert (taken_soft == 1000 + delta) == (abs(delta) < tau), (alpha, delta)


def test_ste_forward_is_hard_in_float32():
    ste = lib().ovcs_soft_ste
    rng = np.random.default_rng(3)
    for _ in range(2000):
        hard = float(rng.integers(0, 65536)); soft = float(np.float32(rng.uniform(-70000, 70000)))
        assert round(ste(soft, hard)) == hard                                 # eq. (4)/(9)/(12): forward value is the hard one


@pytest.mark.parametrize("cfg,T", [(2, 0.1), (3, 1.0), (4, 10.0)])
def test_theorem1_soft_forward_equals_hard(cfg, T):
    """PAPER.md L140 Theorem 1 / L320 Theorem 3: x_t^S == x_t^H for every t, any finite alpha and T."""
    w = make_workload(cfg, batch=4, n_roms=4) if cfg == 4 else make_workload(cfg, batch=3)
    h = OracleVCS(w.roms, w.seeds, w.env_rom); s = OracleVCS(w.roms, w.seeds, w.env_rom)
    acts = w.actions(0, 3)
    for t in range(3):
        h.step(acts[t], 4)
        out = s.step_soft(acts[t], 4, T, 2.0 + 4 * t, threads=os.cpu_count() or 1)
        assert (h.ram() == s.ram()).all() and (h.screen() == s.screen()).all()
        hr, sr = h.regs(), s.regs()
        assert all((hr[f] == sr[f]).all() for f in hr.dtype.names)
        assert (out[:, 6] == 0).all()                                          # no STE/hard mismatch anywhere
        assert (out[:, 3] > 10000).all() and (out[:, 4] > 0).all() and (out[:, 5] > 0).all()
        if T <= 0.1:
            assert (out[:, 7] < 0.03).all()                                    # 510 e^{-10}: the relaxed read barely moves
        else:
            assert (out[:, 7] > 1.0).all()                                     # at T >= 1 the raw relaxed read is far off; STE restores it
        assert ((out[:, 2] > 0) & (out[:, 2] < out[:, 5])).all()              # gates lie strictly inside (0, 1)
