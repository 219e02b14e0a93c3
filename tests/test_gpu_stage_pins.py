"""-m gpu stage pins (SURVEY.md §8(c) "Stage pins for GPU kernels"): every stage of the CUDA path against a
restatement of ITS OWN definition written here (mpmath / numpy; nothing from oracle/ except where the oracle's
exact sums are the input), through the debug exports of include/ls.h.  End-to-end parity would also pass with a
compensating pair of errors in two stages; these cannot.

  P0   1 / psihat(k')                      vs mpmath.quad of (w/2) int phi(z) cos(pi w k' z / n) dz
  K2   (cell, fraction) coordinate, phasor vs 50-digit arithmetic on sampled points, JD-sized offsets too
       (the error floor N_f eps_mach is why the coordinate is carried as an integer plus a fraction)
  K3   bin_start / sorted slots            vs numpy.bincount of exactly computed cells; the sort is a permutation
  K4   fine grid                           vs a numpy restatement of b_l = sum_j c_j psi(l - u_j), and mass conservation
  K5+K6 assembly                           fed the ORACLE's exact sums (Eq. 1) -> power within rounding
"""
import numpy as np
import pytest

from gpu_util import require_cuda
from paper_2409_08090_b200.workloads import Workload, scaled_workload

pytestmark = pytest.mark.gpu
mp = pytest.importorskip("mpmath")
mp.mp.dps = 50


def _plan_and_execute(w, **opts):
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    dev = torch.device("cuda:0")
    t = torch.from_numpy(np.ascontiguousarray(w.t)).to(dev)
    y = torch.from_numpy(np.ascontiguousarray(w.y)).to(dev)
    dy = torch.from_numpy(np.ascontiguousarray(w.dy)).to(dev)
    P = torch.empty((w.batch, w.Nf), dtype=torch.float64, device=dev)
    plan = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, B.LS_F64, w.batch, **opts)
    plan.execute(t, y, dy, P, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return plan, (t, y, dy, P)


def _exact_coords(w, n, width, js, doubled):
    """(l0, eta, phase of f_c t) of input points js, in 50-digit arithmetic on the doubles as given."""
    ndf = mp.mpf(n) * mp.mpf(w.df)
    fc = mp.mpf(w.f0) + mp.mpf(w.Nf // 2) * mp.mpf(w.df)
    out = []
    for j in js:
        tj = mp.mpf(float(w.t[j]))
        u = ndf * tj
        if doubled:
            u = 2 * u
        u = u - mp.floor(u / n) * n                     # folded into [0, n)
        c = int(mp.floor(u))
        f = u - c
        i0 = int(mp.ceil(f - mp.mpf(width) / 2))
        ph = fc * tj
        ph = ph - mp.floor(ph)
        if doubled:
            ph = 2 * ph
        out.append((c + i0, float(2 * (i0 - f) + (width - 1)), float(mp.cos(2 * mp.pi * ph)), float(mp.sin(2 * mp.pi * ph)), c))
    return out


@pytest.mark.parametrize("offset", [0.0, 2450000.5])
def test_K2_coordinates_and_phasors_against_mpmath(offset):
    """1000 sampled points of a config-3-like series (f t up to 2.5e6 cycles; with the Julian-date offset 6e8):
    first touched cell exact, cell fraction to 1e-13 cell, phasor to 1e-12 of its modulus."""
    from paper_2409_08090_b200 import binding as B
    w0 = scaled_workload(3, 200_000)
    w = Workload(w0.name, w0.t + offset, w0.y, w0.dy, w0.f0, w0.df, w0.Nf, "f64", w0.eps)
    plan, _ = _plan_and_execute(w)
    try:
        info = plan.info
        n, width = info["n"], info["w"]
        wn = w.dy.astype(np.float64) ** -2.0
        wn /= wn.sum()
        rng = np.random.default_rng(5)
        js = rng.choice(w.Nd, 1000, replace=False)
        for pset, doubled in ((0, False), (1, True)):
            rec = B.ls_debug_points(plan.handle, w.Nd, pset)
            order = np.argsort(rec[:, 1], kind="stable")
            l0s = rec[order, 1]
            worst_eta = worst_q = 0.0
            for j, (l0, eta, cq, sq, _) in zip(js, _exact_coords(w, n, width, js, doubled)):
                lo, hi = np.searchsorted(l0s, l0), np.searchsorted(l0s, l0, side="right")
                assert hi > lo, (j, l0)                          # the first touched cell is EXACT
                cand = rec[order[lo:hi]]
                best = cand[np.argmin(np.abs(cand[:, 0] - eta))]
                worst_eta = max(worst_eta, abs(best[0] - eta))
                worst_q = max(worst_q, np.hypot(best[2] - wn[j] * cq, best[3] - wn[j] * sq) / wn[j])
            assert worst_eta <= 2e-13, worst_eta                 # eta = 2 x (cell fraction): 1e-13 cell
            assert worst_q <= 1e-12, worst_q
    finally:
        plan.close()


def test_K3_bin_sort_is_a_permutation_in_bin_order():
    from paper_2409_08090_b200 import binding as B
    w = scaled_workload(2, 6000)
    plan, _ = _plan_and_execute(w)
    try:
        info = plan.info
        n, width = info["n"], info["w"]
        nbins = (n + 63) // 64
        js = np.arange(w.Nd)
        for pset, doubled in ((0, False), (1, True)):
            exact = _exact_coords(w, n, width, js, doubled)
            cells = np.array([e[4] for e in exact])
            start = B.ls_debug_bins(plan.handle, nbins, pset)
            expect = np.concatenate([[0], np.cumsum(np.bincount(cells // 64, minlength=nbins))])
            assert np.array_equal(start, expect)
            rec = B.ls_debug_points(plan.handle, w.Nd, pset)
            # a permutation of the input: the multiset of (first touched cell) is the expected one ...
            assert np.array_equal(np.sort(rec[:, 1].astype(np.int64)), np.sort(np.array([e[0] for e in exact])))
            # ... and every record sits inside its own bin: the point's cell is l0 - i0, with i0 = ceil(f - w/2) read off
            # eta = 2 (i0 - f) + (w - 1): eta > 0 (odd w) / eta > -1 (even w) <=> the larger of the two possible i0
            i0 = -(width // 2) + (rec[:, 0] > (0.0 if width % 2 else -1.0))
            cell = (rec[:, 1].astype(np.int64) - i0) % n
            slot_bin = np.searchsorted(start, np.arange(w.Nd), side="right") - 1
            assert np.array_equal(cell // 64, slot_bin)
            assert np.all(np.diff(start) >= 0) and start[-1] == w.Nd
    finally:
        plan.close()


def _es(z, beta):
    return np.exp(beta * (np.sqrt(np.maximum(0.0, 1.0 - z * z)) - 1.0))


def test_P0_deconvolution_table_against_mpmath_quad():
    from paper_2409_08090_b200 import binding as B
    w = scaled_workload(2, 3000)
    plan, _ = _plan_and_execute(w)
    try:
        info = plan.info
        n, width, beta = info["n"], info["w"], mp.mpf(info["beta"])
        ks = np.array([0, 1, w.Nf // 4, w.Nf // 2 - 1, w.Nf // 2])
        got = B.ls_debug_dinv(plan.handle, ks)
        for k, g in zip(ks, got):
            a = mp.pi * width * int(k) / n
            psihat = width * mp.quad(lambda z: mp.exp(beta * (mp.sqrt(1 - z * z) - 1)) * mp.cos(a * z), [0, 0.5, 0.9, 1])
            assert abs(g * psihat - 1) <= 1e-11, (k, float(g * psihat - 1))
    finally:
        plan.close()


def test_K4_fine_grid_against_numpy_restatement_and_mass_conservation():
    """n = 2^16 (every tile is written): the three fine grids as the spreading kernel left them against
    b_l = sum_j c_j psi(l - u_j), psi(s) = exp(beta (sqrt(1 - (2 s / w)^2) - 1)), l mod n."""
    from paper_2409_08090_b200 import binding as B
    w = scaled_workload(2, 3000)
    plan, (t, y, dy, _) = _plan_and_execute(w, no_autotune=1)
    try:
        info = plan.info
        n, width, beta = info["n"], info["w"], info["beta"]
        assert n == 1 << 16
        wn = w.dy.astype(np.float64) ** -2.0
        wn /= wn.sum()
        ybar = float(np.sum(wn * w.y[0]))
        psihat0 = 1.0 / B.ls_debug_dinv(plan.handle, [0])[0]
        js = np.arange(w.Nd)
        for slot, doubled, strength in ((0, True, wn), (1, False, wn), (2, False, wn * (w.y[0] - ybar))):
            grid = B.ls_debug_grid(plan.handle, n, t, y, dy, slot)
            ref = np.zeros(n, dtype=np.complex128)
            for j, (l0, eta, cq, sq, _) in zip(js, _exact_coords(w, n, width, js, doubled)):
                x0 = (eta - (width - 1)) / 2.0                   # l0 - u_j, in [-w/2, -w/2 + 1)
                s = x0 + np.arange(width)
                ref[(l0 + np.arange(width)) % n] += strength[j] * (cq + 1j * sq) * _es(2.0 * s / width, beta)
            err = np.linalg.norm(grid - ref) / np.linalg.norm(ref)
            assert err <= 5e-12, (slot, err)                     # the kernel is a degree-12 piecewise polynomial: <= 7e-13
            c_sum = np.sum([strength[j] * (e[2] + 1j * e[3]) for j, e in zip(js, _exact_coords(w, n, width, js, doubled))])
            assert abs(grid.sum() / c_sum - psihat0) <= 1e-8 * psihat0   # sum_l psi(l - u) = psihat(0) (1 + O(eps))
    finally:
        plan.close()


@pytest.mark.parametrize("no_float,norm", [(0, 0), (1, 0), (0, 3)])
def test_K6_assembly_fed_the_oracles_exact_sums(no_float, norm):
    import oracle
    from paper_2409_08090_b200 import binding as B
    require_cuda()
    w = scaled_workload(2, 2000)
    _, sums, _ = oracle.direct(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, return_sums=True)
    W, ybar, YY = oracle.stats(w.y[0], w.dy)
    got = B.ls_debug_assemble(sums, YY, W, no_float, norm)
    s2 = sums.copy()
    if no_float:
        s2[:, 2:4] = 0.0                                         # fixed mean: the (S, C) sums of the weights drop out
    Po = oracle.assemble(s2, YY)[0]
    if norm == 3:
        Po = 0.5 * Po * W * YY                                   # psd normalisation (A19)
    assert np.max(np.abs(got - Po) / np.maximum(np.abs(Po), 1e-300)) <= 1e-12
