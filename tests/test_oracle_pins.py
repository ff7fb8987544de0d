"""Pins of the CPU oracle against things other than itself (paper identities, closed forms,
quadrature, brute force, published RNG vectors).  CPU only (-m "not gpu").

Each test names the passage of PAPER.md (or the DESIGN.md reading) it checks.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1609_07936_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
TWO_PI = 2.0 * math.pi


# ----------------------------------------------------------------------------- Philox (G14)
def _py_philox(ctr, key):
    """Independent restatement of Philox4x32-10 (python integers)."""
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l[0] not in "#\n"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_random_counters_match_python_restatement():
    rng = np.random.default_rng(0)
    for _ in range(50):
        ctr = [int(x) for x in rng.integers(0, 2**32, 4)]
        key = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert [int(x) for x in oracle.philox4x32_10(ctr, key)] == _py_philox(ctr, key)


# ----------------------------------------------------------------------------- O1 kernel table
def test_kernel_table_equals_quadrature_of_rectangle():
    """Eq. 5-6: K[k][j] = (1/2pi) int_bin exp(-w tau_j) dw.  Non-square grid so a
    transposed table fails."""
    omega = np.arange(7) * 0.37          # left edges
    tau = np.arange(5) * 0.21
    K = oracle.kernel_table(omega, tau)
    assert K.shape == (7, 5)
    dw = 0.37
    for k in range(7):
        for j in range(5):
            ref, _ = integrate.quad(lambda w: math.exp(-w * tau[j]) / TWO_PI, omega[k], omega[k] + dw,
                                    epsabs=0, epsrel=2e-14)
            assert K[k, j] == pytest.approx(ref, rel=2e-14)


def test_c_vector_eq8_and_small_argument():
    """Eq. 8: c_0 = dw/2pi; c_i = (1-exp(-i dw dtau))/(2pi i dtau).  At small x the
    expm1 form (reading G2) must agree with the series to full precision."""
    omega = np.arange(16) * 0.005859375
    tau = np.array([0.0, 0.01, 0.02, 5.11])
    c = oracle.cvec(omega, tau)
    dw = 0.005859375
    assert c[0] == pytest.approx(dw / TWO_PI, rel=1e-15)
    for j in (1, 2, 3):
        x = dw * tau[j]
        series = (dw / TWO_PI) * (1 - x / 2 + x * x / 6 - x**3 / 24 + x**4 / 120 - x**5 / 720)
        assert c[j] == pytest.approx(series, rel=3e-15)


def test_flat_spectrum_closed_form_and_eq16():
    """a == 1 on [0, w_max]: M(tau) = (1 - exp(-w_max tau))/(2 pi tau); Eq. 16: M(0) = c_0 A."""
    n_omega, w_max = 40, 5.0
    omega = np.arange(n_omega) * (w_max / n_omega)
    tau = np.arange(9) * 0.3
    K = oracle.kernel_table(omega, tau)
    M = oracle.forward(K, np.ones(n_omega))
    ref = np.where(tau > 0, -np.expm1(-w_max * np.maximum(tau, 1e-300)) / (TWO_PI * np.maximum(tau, 1e-300)),
                   w_max / TWO_PI)
    np.testing.assert_allclose(M, ref, rtol=1e-14)
    a = np.random.default_rng(1).random(n_omega)
    assert oracle.forward(K, a)[0] == pytest.approx((w_max / n_omega) / TWO_PI * a.sum(), rel=1e-15)


# ----------------------------------------------------------------------------- O2 forward
def test_forward_matches_longdouble_piecewise_integral():
    """Eq. 5: the model is the exact integral of the piecewise-constant function —
    evaluated here bin by bin in extended precision without the c_j q^{ij} factorisation."""
    omega = np.arange(64) * 0.125
    tau = np.arange(32) * 0.05
    a = wl.bin_averages(omega, 0.125)
    M = oracle.forward(oracle.kernel_table(omega, tau), a)
    al, ol = a.astype(np.longdouble), omega.astype(np.longdouble)
    dw = np.longdouble(0.125)
    two_pi = 2 * np.longdouble(np.pi) + np.longdouble(2.4492935982947064e-16)  # pi to ~1e-32
    for j, t in enumerate(tau.astype(np.longdouble)):
        if t == 0:
            ref = (al * dw).sum() / two_pi
        else:
            ref = (al * (np.exp(-ol * t) - np.exp(-(ol + dw) * t)) / t).sum() / two_pi
        assert float(abs(M[j] - ref) / ref) < 1e-13


def test_forward_converges_to_simpson_F_second_order():
    """north_star check: with a = exact bin averages of the truncated double Lorentzian the model tends
    to the 1e6-interval Simpson F with error ~ domega^2 (ratio 4 per halving)."""
    tau = np.arange(16) * 0.1
    F = wl.correlation_simpson(tau, 1_000_000)
    errs = []
    for n in (256, 512, 1024, 2048):
        dw = 8.0 / n
        omega = np.arange(n) * dw
        M = oracle.forward(oracle.kernel_table(omega, tau), wl.bin_averages(omega, dw))
        errs.append(np.abs(M - F)[1:].max())
        assert abs(M[0] - F[0]) < 1e-13            # tau = 0: both are (1/2pi) int S exactly
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(3.8 < r < 4.2 for r in ratios), ratios
    assert errs[-1] < 1e-6


# ----------------------------------------------------------------------------- O3 residue
def test_chi2_brute_force_tiny_grid():
    """Eq. 9 with sigma (G3), on a 3x4 grid where the model is integrated numerically."""
    omega = np.array([0.0, 0.5, 1.0])
    tau = np.array([0.0, 0.4, 0.8, 1.2])
    a = np.array([0.3, 1.1, 0.6])
    F = np.array([0.16, 0.11, 0.08, 0.055])
    sigma = np.array([1e-2, 2e-2, 1e-2, 3e-2])
    M = oracle.forward(oracle.kernel_table(omega, tau), a)
    brute = 0.0
    for j in range(4):
        m = sum(integrate.quad(lambda w: a[k] * math.exp(-w * tau[j]) / TWO_PI, omega[k], omega[k] + 0.5,
                               epsabs=0, epsrel=2e-14)[0] for k in range(3))
        brute += ((m - F[j]) / sigma[j]) ** 2
    assert oracle.chi2(M, F, sigma) == pytest.approx(brute, rel=1e-12)
    assert oracle.chi2(M, F, None) == pytest.approx(((M - F) ** 2).sum(), rel=1e-14)


# ----------------------------------------------------------------------------- O4 start
def test_init_tilt_meets_both_sum_rules_and_is_positive():
    for name in ("tiny", "small"):
        w = wl.make(name, simpson_intervals=20_000)
        a = oracle.init_tilt(w.omega, w.A, w.B)
        wm = w.omega + 0.5 * w.domega
        assert (a > 0).all()
        assert a.sum() == pytest.approx(w.A, rel=1e-13)
        assert (a * wm).sum() == pytest.approx(w.B, rel=1e-12)
    # reduces to the flat spectrum when omega_c is the grid midpoint (G4)
    omega = np.arange(10) * 0.2
    a = oracle.init_tilt(omega, 5.0, 5.0 * 1.0)
    np.testing.assert_allclose(a, 0.5, rtol=1e-12)
    with pytest.raises(ValueError):
        oracle.init_tilt(omega, 1.0, 100.0)


# ----------------------------------------------------------------------------- O5 move
def _oracle_for(w, seed=1234, **kw):
    o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, seed, **kw)
    return o


@pytest.fixture(scope="module")
def tiny():
    return wl.make("tiny", simpson_intervals=100_000)


def test_move_draws_follow_the_counter_layout(tiny):
    """Reading G14/G11/G6: ctr = (walker, sweep, move, 0); p = (x0 N)>>32, s != p; rho = 1 - y eta (2u-1)."""
    o = _oracle_for(tiny, seed=0x1234_5678_9ABC_DEF0)
    o.init_walkers(4)
    for (wk, sw, mv) in [(0, 0, 0), (3, 17, 63), (2, 100000, 5)]:
        tr = o.move(wk, sw, mv, T=1.0, y=0.5)
        x = _py_philox([wk, sw, mv, 0], [0x9ABCDEF0, 0x12345678])
        p = (x[0] * 64) >> 32
        s = (x[1] * 63) >> 32
        s += s >= p
        assert (tr["p"], tr["s"]) == (p, s) and p != s
        rho = 1.0 - 0.5 * tiny.eta * (2.0 * ((x[2] + 0.5) / 2**32) - 1.0)
        assert tr["rho"] == pytest.approx(rho, rel=1e-15)
        assert tr["ln_u"] == pytest.approx(math.log((x[3] + 0.5) / 2**32), rel=1e-15)


def test_index_selection_uniform(tiny):
    """Zero-length walk = uniform p and uniform s != p."""
    o = _oracle_for(tiny)
    o.init_walkers(1)
    tr, _ = o.anneal(np.full(300, 1.0), trace_walkers=(0, 1))
    p, s = tr["p"].ravel(), tr["s"].ravel()
    assert (p != s).all() and p.min() == 0 and p.max() == 63 and s.min() == 0 and s.max() == 63
    n = p.size
    for v in (p, s):
        cnt = np.bincount(v, minlength=64)
        chi = ((cnt - n / 64) ** 2 / (n / 64)).sum()
        assert chi < 63 + 5 * math.sqrt(2 * 63)
    assert np.bincount((s - p) % 64, minlength=64)[0] == 0


def test_move_preserves_both_sum_rules_and_tau0(tiny):
    """Eq. 20-21: A and B unchanged to 1e-13 per move; Eq. 16: dM_0 = 0."""
    o = _oracle_for(tiny)
    o.init_walkers(8)
    wm = tiny.omega + 0.5 * tiny.domega
    n_acc = 0
    for mv in range(400):
        for wk in range(8):
            a0, M0 = o.a[wk].copy(), o.M[wk].copy()
            tr = o.move(wk, 0, mv, T=1e300)         # T -> inf: every feasible move is accepted
            if tr["flags"] & 2:
                n_acc += 1
                assert abs(o.a[wk].sum() - a0.sum()) <= 1e-13 * a0.sum()
                assert abs((o.a[wk] * wm).sum() - (a0 * wm).sum()) <= 1e-13 * (a0 * wm).sum()
                assert abs(o.M[wk][0] - M0[0]) <= 4e-16 * M0[0]
                assert (o.a[wk] >= 0).all()
            else:
                assert not (tr["flags"] & 1)         # at T=inf only infeasible moves are rejected
                np.testing.assert_array_equal(o.a[wk], a0)
                np.testing.assert_array_equal(o.M[wk], M0)
    assert n_acc > 1000


def test_move_is_a_homothety_about_the_two_bin_vertex(tiny):
    """Derived from Eq. 17-21: a' - e = rho (a - e), e = two-bin spectrum carrying A and B in bins p, s."""
    o = _oracle_for(tiny)
    o.init_walkers(1)
    wm = tiny.omega + 0.5 * tiny.domega
    A, B = tiny.A, tiny.B
    done = 0
    for mv in range(200):
        a0 = o.a[0].copy()
        tr = o.move(0, 3, mv, T=1e300)
        if not tr["flags"] & 2:
            continue
        p, s, rho = tr["p"], tr["s"], tr["rho"]
        e = np.zeros_like(a0)
        e[p] = (B - A * wm[s]) / (wm[p] - wm[s])
        e[s] = (B - A * wm[p]) / (wm[s] - wm[p])
        np.testing.assert_allclose(o.a[0] - e, rho * (a0 - e), rtol=0, atol=1e-12 * np.abs(e).max())
        done += 1
    assert done > 50


def test_straddling_contraction_is_never_infeasible(tiny):
    """If p, s straddle omega_c = B/A (e >= 0) and 0 < rho <= 1 the move is a convex combination
    (PAPER.md:137-143 + homothety): positivity can never fail."""
    o = _oracle_for(tiny)
    o.init_walkers(1)
    wm = tiny.omega + 0.5 * tiny.domega
    wc = tiny.B / tiny.A
    seen = 0
    for sw in range(40):
        for mv in range(64):
            tr = o.move(0, sw, mv, T=1e-300)        # nothing uphill accepted, state nearly frozen
            straddle = (wm[tr["p"]] - wc) * (wm[tr["s"]] - wc) < 0
            if straddle and tr["rho"] <= 1.0:
                assert tr["flags"] & 1
                seen += 1
    assert seen > 100


def test_incremental_dchi2_equals_from_scratch(tiny):
    """Eq. 22 with c_j (reading G1) + Eq. 9: Delta chi^2 and the updated M agree with a full recompute."""
    o = _oracle_for(tiny)
    o.init_walkers(2)
    K = o.K
    for mv in range(300):
        wk = mv % 2
        a0 = o.a[wk].copy()
        c0 = oracle.chi2(oracle.forward(K, a0), tiny.F, tiny.sigma)
        tr = o.move(wk, 1, mv, T=1e300)
        if tr["flags"] & 2:
            M1 = oracle.forward(K, o.a[wk])
            c1 = oracle.chi2(M1, tiny.F, tiny.sigma)
            np.testing.assert_allclose(o.M[wk], M1, rtol=1e-12)
            assert abs((c1 - c0) - tr["dchi2"]) <= 1e-12 * tr["l1"] + 1e-9 * abs(tr["dchi2"])


def test_move_brute_force_on_tiny_grid():
    """north_star: brute-force chi^2 on tiny grids — the move's Delta chi^2 against chi^2 evaluated by
    numerical integration of the rectangles before and after."""
    omega = np.arange(4) * 0.6
    tau = np.arange(3) * 0.5
    a = np.array([0.9, 0.4, 0.7, 0.2])
    wm = omega + 0.3
    A, B = a.sum(), (a * wm).sum()
    F = np.array([0.2, 0.12, 0.08])
    sigma = np.array([0.01, 0.02, 0.015])

    def brute(av):
        tot = 0.0
        for j in range(3):
            m = sum(integrate.quad(lambda w: av[k] * math.exp(-w * tau[j]) / TWO_PI, omega[k], omega[k] + 0.6,
                                   epsabs=0, epsrel=2e-14)[0] for k in range(4))
            tot += ((m - F[j]) / sigma[j]) ** 2
        return tot

    o = oracle.Oracle(omega, tau, F, sigma, A, B, 0.3, 99)
    o.init_walkers(1, spectra=a[None, :])
    n = 0
    for mv in range(30):
        a0 = o.a[0].copy()
        tr = o.move(0, 0, mv, T=1e300)
        if tr["flags"] & 2:
            assert brute(o.a[0]) - brute(a0) == pytest.approx(tr["dchi2"], rel=1e-9, abs=1e-9)
            n += 1
    assert n >= 10


# ----------------------------------------------------------------------------- Metropolis (Eq. 10)
def test_metropolis_limits(tiny):
    o = _oracle_for(tiny)
    o.init_walkers(4)
    c_prev = o.chi2.copy()
    _, flags = o.anneal(np.full(5, 1e-300), want_flags=True)     # T -> 0+: chi^2 never increases
    assert (o.chi2 <= c_prev).all()
    tr, flags = o.anneal(np.full(3, 1e300), trace_walkers=(0, 4), want_flags=True)  # T -> inf
    assert ((flags & 1) * 2 == (flags & 2)).all()                  # feasible <=> accepted
    assert (tr["flags"] == flags[:, :, :]).all()


def test_metropolis_frequency_matches_boltzmann_factor(tiny):
    """Acceptance frequency of uphill moves in a Delta/T bin equals exp(-Delta/T)."""
    o = _oracle_for(tiny, amp_mode=0)
    o.init_walkers(64)
    o.anneal(np.full(30, 1e3))                                     # relax away from the start
    keep = (o.a.copy(), o.M.copy(), o.chi2.copy(), o.sweep)
    tr, _ = o.anneal(np.full(10, 1e3), trace_walkers=(0, 64))      # probe the scale of uphill moves
    t = tr.ravel()
    up = ((t["flags"] & 1) == 1) & (t["dchi2"] > 0)
    T = float(np.median(t["dchi2"][up]))
    o.a[:], o.M[:], o.chi2[:], o.sweep = keep
    tr, _ = o.anneal(np.full(80, T), trace_walkers=(0, 64))
    t = tr.ravel()
    feas = (t["flags"] & 1) == 1
    x = t["dchi2"] / T
    for lo, hi in [(0.05, 0.15), (0.3, 0.5), (0.9, 1.1), (1.8, 2.2)]:
        sel = feas & (x > lo) & (x < hi)
        n = sel.sum()
        assert n > 300, (lo, hi, n)
        expect = np.exp(-x[sel]).mean()
        got = ((t["flags"][sel] & 2) == 2).mean()
        assert abs(got - expect) < 5 * math.sqrt(expect * (1 - expect) / n), (lo, hi, got, expect)
    down = feas & (x < 0)
    assert ((t["flags"][down] & 2) == 2).all()                     # downhill always accepted


# ----------------------------------------------------------------------------- Eq. 30
def test_amp_factor_eq30():
    """y = 1 for a >= p; (a/p)^m below; p = 1, m = 2 gives y = a^2."""
    assert oracle.amp_factor(1.0) == 1.0
    assert oracle.amp_factor(0.5) == 0.25
    assert oracle.amp_factor(0.25, amp_p=0.5, amp_m=3.0) == pytest.approx(0.125)
    assert oracle.amp_factor(0.7, amp_p=0.5) == 1.0
    assert oracle.amp_factor(0.0) == 1e-6                          # floor (G7)


def test_sweep_updates_y_from_its_own_acceptance(tiny):
    o = _oracle_for(tiny)
    o.init_walkers(3)
    _, flags = o.anneal(np.array([0.5]), want_flags=True)
    rate = ((flags[:, 0, :] & 2) == 2).sum(axis=1) / 64.0
    np.testing.assert_allclose(o.y, np.where(rate >= 1, 1.0, np.maximum(rate**2, 1e-6)), rtol=1e-15)
    assert (o.acc == ((flags & 2) == 2).sum(axis=(1, 2))).all()


# ----------------------------------------------------------------------------- resync / splitting
def test_split_runs_and_resync_are_consistent(tiny):
    """Absolute sweep counter: one 6-sweep call == 2+4 sweeps; resync leaves chi^2 to rounding."""
    sched = wl.geometric_schedule(1.0, 0.1, 6)
    o1 = _oracle_for(tiny); o1.init_walkers(4); o1.anneal(sched)
    o2 = _oracle_for(tiny); o2.init_walkers(4); o2.anneal(sched[:2]); o2.anneal(sched[2:])
    np.testing.assert_array_equal(o1.a, o2.a)
    np.testing.assert_array_equal(o1.chi2, o2.chi2)
    c = o1.chi2.copy()
    o1.resync()
    np.testing.assert_allclose(o1.chi2, c, rtol=1e-9)


# ----------------------------------------------------------------------------- O8 branching
def test_branch_multipliers_sum_to_W_and_have_mean_w(tiny):
    """Eq. 25: E[m] = w and sum m = W for the once-generated xi set (comb, B2)."""
    o = _oracle_for(tiny)
    o.init_walkers(64)
    o.anneal(np.full(3, 1.0))
    T = float(np.std(o.chi2)) * 2.0
    w = np.exp(-(o.chi2 - o.chi2.min()) / T)
    w *= 64 / w.sum()
    acc = np.zeros(64)
    a_keep, M_keep, c_keep = o.a.copy(), o.M.copy(), o.chi2.copy()
    n_ev = 400
    for ev in range(n_ev):
        o.a[:], o.M[:], o.chi2[:] = a_keep, M_keep, c_keep
        o.sweep = 1000 + ev                                       # xi depends on the sweep counter
        n_rec, mult, donor = o.branch(T, 0.0)                     # t = 0: state untouched
        assert mult.sum() == 64
        assert ((mult == np.floor(w)) | (mult == np.ceil(w)) | (np.abs(mult - w) < 1 + 1e-9)).all()
        assert n_rec == (mult == 0).sum() == np.maximum(mult - 1, 0).sum()
        acc += mult
        np.testing.assert_array_equal(o.a, a_keep)                # t = 0 is a no-op (Eq. 26)
    np.testing.assert_allclose(acc / n_ev, w, atol=5 * 0.5 / math.sqrt(n_ev) + 1e-9)


def test_branch_imprint_t1_copies_and_t_preserves_sum_rules(tiny):
    """Eq. 26: t = 1 is classic branching (recipient == donor); any t keeps A, B
    (linearity); donors unchanged; chi^2 of recipients recomputed from their new spectrum."""
    wm = tiny.omega + 0.5 * tiny.domega
    for t in (1.0, 0.1):
        o = _oracle_for(tiny)
        o.init_walkers(64)
        o.anneal(np.full(3, 1.0))
        a0 = o.a.copy()
        n_rec, mult, donor = o.branch(float(np.std(o.chi2)), t)
        assert n_rec > 0
        rec = np.where(donor >= 0)[0]
        assert (mult[rec] == 0).all() and (mult[donor[rec]] >= 2).all()
        # each donor serves exactly m-1 recipients, recipients in ascending order get ascending donors
        assert (np.bincount(donor[rec], minlength=64) == np.maximum(mult - 1, 0)).all()
        assert (np.diff(donor[rec]) >= 0).all()
        others = np.where(donor < 0)[0]
        np.testing.assert_array_equal(o.a[others], a0[others])
        for i in rec:
            if t == 1.0:
                np.testing.assert_array_equal(o.a[i], a0[donor[i]])
            np.testing.assert_allclose(o.a[i], t * a0[donor[i]] + (1 - t) * a0[i], rtol=1e-15)
            assert o.a[i].sum() == pytest.approx(tiny.A, rel=1e-13)
            assert (o.a[i] * wm).sum() == pytest.approx(tiny.B, rel=1e-12)
            M = oracle.forward(o.K, o.a[i])
            np.testing.assert_array_equal(o.M[i], M)
            assert o.chi2[i] == oracle.chi2(M, tiny.F, tiny.sigma)


# ----------------------------------------------------------------------------- regression fixture
def test_oracle_reproduces_its_committed_trace():
    """tests/golden/oracle_tiny_trace.txt is written by tests/golden/make_oracle_golden.py from the oracle alone;
    integer fields must match exactly, floating fields to 1e-13 (libm exp/log may differ in the last bit
    between machines)."""
    sys_path = os.path.join(GOLDEN, "make_oracle_golden.py")
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_oracle_golden", sys_path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    _, chi2_0, tr, o = mod.compute()
    n = 0
    for line in open(os.path.join(GOLDEN, "oracle_tiny_trace.txt")):
        if line.startswith("# chi2_0"):
            vals = [float(x) for x in line.split()[2:]]
            np.testing.assert_allclose(chi2_0, vals, rtol=1e-12)
        if line.startswith("#"):
            continue
        f = line.split()
        wk, sw, m = int(f[0]), int(f[1]), int(f[2])
        t = tr[wk, sw, m]
        assert (t["p"], t["s"], t["flags"]) == (int(f[3]), int(f[4]), int(f[5]))
        for name, val in zip(("rho", "delta_p", "delta_s", "dchi2", "ln_u"), f[6:11]):
            assert float(t[name]) == pytest.approx(float(val), rel=1e-11, abs=1e-300), name
        n += 1
    assert n == 96


# ---- O9 smoothing, Eq. 27-29 ------------------------------------------------------
def test_stencil_cosine_modes_are_eigenvectors():
    """Eq. 27-29 is the 3-point diffusion stencil with reflecting ends: the DCT-II modes cos(pi n (j + 1/2) / N) are
    its eigenvectors with eigenvalue 1 - 2 s (1 - cos(pi n / N)) (a textbook fact, not the oracle's own formula)."""
    N, s = 48, 0.037
    j = np.arange(N)
    for n in (0, 1, 5, 17, N - 1):
        mode = np.cos(np.pi * n * (j + 0.5) / N)
        lam = 1.0 - 2.0 * s * (1.0 - math.cos(math.pi * n / N))
        np.testing.assert_allclose(oracle.stencil(mode, s), lam * mode, rtol=0, atol=2e-15)


def test_stencil_is_not_transposed_or_shifted_and_s0_is_identity():
    """A single spike spreads s to each neighbour (and keeps 1 - s at an end bin); s = 0 changes nothing."""
    N, s = 9, 0.25
    for k in range(N):
        e = np.zeros(N); e[k] = 1.0
        want = np.zeros(N)
        want[k] = 1 - 2 * s if 0 < k < N - 1 else 1 - s
        if k > 0: want[k - 1] = s
        if k < N - 1: want[k + 1] = s
        np.testing.assert_allclose(oracle.stencil(e, s), want, rtol=0, atol=1e-16)
    a = np.random.default_rng(3).random(N)
    np.testing.assert_array_equal(oracle.stencil(a, 0.0), a)
    ramp = np.arange(N, dtype=float)
    np.testing.assert_allclose(oracle.stencil(ramp, s)[1:-1], ramp[1:-1], rtol=1e-15)   # interior of a linear ramp


def test_stencil_keeps_first_sum_rule_and_shifts_the_second_as_the_paper_says():
    """:197 — the first sum rule is preserved, the second violated 'of the order of s (a_{N-1} - a_0) / N': exactly
    sum_j w_j (a'_j - a_j) = s domega (a_0 - a_{N-1}) for bin midpoints w_j (summation by parts)."""
    rng = np.random.default_rng(5)
    N, s, dw = 64, 0.03, 0.125
    wm = (np.arange(N) + 0.5) * dw
    for _ in range(5):
        a = rng.random(N) + 0.01
        b = oracle.stencil(a, s)
        assert abs(b.sum() - a.sum()) <= 1e-14 * a.sum()
        assert abs(((b - a) * wm).sum() - s * dw * (a[0] - a[-1])) <= 1e-13 * (a * wm).sum()


def test_smooth_restores_both_sum_rules_keeps_positivity_and_resyncs(tiny):
    """Reading S2 (linear tilt about the mean frequency) + resync: A and B back to 1e-13, a > 0, M = forward(a)."""
    o = _oracle_for(tiny)
    o.init_walkers(16)
    o.anneal(tiny.schedule[:5])
    a0 = o.a.copy()
    wm = tiny.omega + 0.5 * tiny.domega
    o.smooth(0.02)
    np.testing.assert_allclose(o.a.sum(axis=1), tiny.A, rtol=1e-13)
    np.testing.assert_allclose((o.a * wm).sum(axis=1), tiny.B, rtol=1e-13)
    assert (o.a > 0).all()
    st = np.array([oracle.stencil(r, 0.02) for r in a0])
    assert np.abs(o.a / st - 1.0).max() < 1e-3                      # the renormalisation is a small correction
    M, c2 = o.M.copy(), o.chi2.copy()
    o.resync()
    np.testing.assert_array_equal(o.M, M)
    np.testing.assert_array_equal(o.chi2, c2)
    o2 = _oracle_for(tiny); o2.init_walkers(16, a0)
    o2.smooth(0.0)                                                   # s = 0: only rounding-level renormalisation
    np.testing.assert_allclose(o2.a, a0, rtol=1e-12)


def test_smooth_clamps_the_tilt_where_it_would_turn_a_coefficient_negative(tiny):
    """Reading S2, positivity branch (PAPER.md:197 "requires an additional renormalization"; Eq. 10, :97, needs
    a_k >= 0).  Weight piled on the last three bins and s = 0.5: the stencil pushes B down by s domega a_{N-1} (:197), the
    variance of such a row is a few domega^2, so the tilt that would restore B has 1 + kappa (w_0 - wbar) < 0 — it would
    make the coefficients of the lowest bins negative.  What the clamp must give, whatever its formula: no negative
    coefficient; the factor 0 (to one rounding, never below) at the end bin it clamps on — kappa is the largest admissible one; sum a
    untouched (a tilt about the mean keeps it for ANY kappa); B moved TOWARDS its target, not away and not past it."""
    n = tiny.n_omega
    wm = tiny.omega + 0.5 * tiny.domega
    rng = np.random.Generator(np.random.Philox(5))
    for row in range(6):
        a = 1e-3 + rng.uniform(0.0, 1e-3, n)
        a[-3:] += rng.uniform(5.0, 10.0, 3)
        A, B = a.sum(), (a * wm).sum()
        o = oracle.Oracle(tiny.omega, tiny.tau, tiny.F, tiny.sigma, A, B, tiny.eta, 1)
        o.init_walkers(1, a[None, :].copy())
        st = oracle.stencil(a, 0.5)
        B_st = (st * wm).sum()
        np.testing.assert_allclose(B_st - B, 0.5 * tiny.domega * (a[0] - a[-1]), rtol=1e-9)     # :197, B fell
        wbar = B_st / A
        V = (st * (wm - wbar) ** 2).sum()
        assert 1.0 + (B - B_st) / V * (wm[0] - wbar) < -0.05                                    # the unclamped tilt is inadmissible
        o.smooth(0.5)
        out = o.a[0]
        assert (out >= 0.0).all()
        # clamped at bin 0: the factor there is 1 + fl(-1/d) d = 0 up to the one rounding of the quotient, from above
        assert 0.0 <= out[0] <= 2.0 ** -52 * st[0] and st[0] > 0.0 and (out[1:] > 0.0).all()
        assert abs(out.sum() - A) <= 1e-14 * A
        B_out = (out * wm).sum()
        assert B_st < B_out < B and (B - B_out) < (B - B_st)                                    # towards B, not past it
        # the factor out_k / st_k is linear in w_k through (w_0, 0) and (wbar, 1)
        np.testing.assert_allclose(out / st, (wm - wm[0]) / (wbar - wm[0]), rtol=0, atol=1e-12)
        np.testing.assert_array_equal(o.M[0], oracle.forward(o.K, out))                         # resynced
    # the mirror image (weight on the first bins): the clamp acts at the last bin
    a = 1e-3 + rng.uniform(0.0, 1e-3, n)
    a[:3] += rng.uniform(5.0, 10.0, 3)
    A, B = a.sum(), (a * wm).sum()
    o = oracle.Oracle(tiny.omega, tiny.tau, tiny.F, tiny.sigma, A, B, tiny.eta, 1)
    o.init_walkers(1, a[None, :].copy())
    st = oracle.stencil(a, 0.5)
    o.smooth(0.5)
    out = o.a[0]
    B_st, B_out = (st * wm).sum(), (out * wm).sum()
    assert (out >= 0.0).all() and out[-1] <= 2.0 ** -52 * st[-1] and abs(out.sum() - A) <= 1e-14 * A
    assert B < B_out < B_st


def test_adaptive_branching_strength_follows_the_acceptance_rate(tiny):
    """Reading B7 (imprinting strength and branching fraction are reduced "according to the decrease of
    the acceptance probability").  What the sentence fixes: full strength while the acceptance has not decreased (the
    block with the largest rate so far), never more than full strength, less when the block's rate is lower, none when
    nothing is accepted.  Then the protocol: a hot block followed by a cold one — the first branches at full strength
    (same state as the run without adaptation), the second with strength and fraction both cut by the ratio of the two
    acceptance rates, so fewer walkers are replaced than without adaptation."""
    f = oracle.branching_strength_scale
    rates = [0.40, 0.42, 0.30, 0.35, 0.05, 0.0]
    best, scales = 0.0, []
    for r in rates:
        best = max(best, r)
        scales.append(f(r, best))
    assert scales[0] == 1.0 and scales[1] == 1.0                      # at the running maximum
    assert all(0.0 <= x <= 1.0 for x in scales)
    assert scales[2] < 1.0 and scales[2] < scales[3] < 1.0 and scales[4] < scales[2] and scales[5] == 0.0
    np.testing.assert_allclose(scales[2:5], np.array(rates[2:5]) / 0.42, rtol=1e-15)
    assert f(0.0, 0.0) == 0.0                                         # nothing accepted yet: no branching at all

    W, k, frac, t = 200, 3, 0.25, 0.5
    hot, cold = 10.0, 1e-9                                            # in units of the starting residue (T_override is absolute)
    o = _oracle_for(tiny); o.init_walkers(W)
    c0 = float(np.mean(o.chi2))
    Ts = [hot * c0, cold * c0]
    o.anneal_selfcool(2, k, n_boil=0, n_ramp=1, t_imprint=t, branch_fraction=frac, adapt=True, T_override=Ts)
    # replay with the public pieces; block 0 at full strength
    r = _oracle_for(tiny); r.init_walkers(W)
    r.anneal(np.full(k, Ts[0]))
    acc0 = int(r.acc.sum())
    plain = _oracle_for(tiny); plain.init_walkers(W)
    plain.anneal_selfcool(1, k, n_boil=0, n_ramp=1, t_imprint=t, branch_fraction=frac, adapt=False, T_override=Ts[:1])
    r.branch_fraction(frac, t)
    np.testing.assert_array_equal(r.a, plain.a)                       # scale = 1 in the first block
    r.anneal(np.full(k, Ts[1]))
    acc1 = int(r.acc.sum()) - acc0
    assert 0 < acc1 < 0.8 * acc0                                      # the cold block accepts less
    scale = acc1 / acc0
    full = _oracle_for(tiny); full.init_walkers(W, r.a.copy()); full.chi2[:] = r.chi2; full.sweep = r.sweep
    _, n_full, _, _ = full.branch_fraction(frac, t)
    before = r.a.copy()
    _, n_cut, mult, donor = r.branch_fraction(frac * scale, t * scale)
    np.testing.assert_array_equal(r.a, o.a)                           # the protocol did exactly this
    assert n_cut < n_full and abs(n_cut - frac * scale * W) <= 0.02 * W + 1
    rec = np.flatnonzero(mult == 0)
    if rec.size:                                                      # imprint strength t * scale (Eq. 26)
        i = rec[0]
        np.testing.assert_allclose(r.a[i], t * scale * before[donor[i]] + (1.0 - t * scale) * before[i], rtol=1e-13)


# ---- f1 self-cooling ------------------------------------------------------------
def test_selfcool_rule_follows_the_papers_statements():
    """What the paper fixes: T starts at 10 starting residues (:216); it sits at chi2_ave while boiling, is ramped
    towards chi2_min, then goes BELOW chi2_min and falls in proportion to the number of steps (:162).  The lengths
    of the phases and the rate are the build's constants (readings C2: unpinned)."""
    f = oracle.selfcool_temperature
    chi0, ave, mn, nb, nr = 3.0e8, 5.0e4, 2.0e3, 3, 4
    assert f(0, chi0, ave, mn, nb, nr) == 10.0 * chi0
    assert all(f(b, chi0, ave, mn, nb, nr) == ave for b in (1, 2, 3))
    ramp = [f(b, chi0, ave, mn, nb, nr) for b in range(nb + 1, nb + nr + 1)]
    assert all(x > y for x, y in zip([ave] + ramp, ramp)) and ramp[-1] == mn and ave > ramp[0] > mn
    np.testing.assert_allclose(np.diff(ramp), (mn - ave) / nr, rtol=1e-12)              # linear
    fr = [f(b, chi0, ave, mn, nb, nr, freeze_rate=0.5) for b in range(nb + nr + 1, nb + nr + 6)]
    assert all(x < mn for x in fr)
    np.testing.assert_allclose([x * (1 + 0.5 * k) for k, x in enumerate(fr, start=1)], mn, rtol=1e-14)   # ~ 1 / steps


def test_selfcool_protocol_runs_blocks_of_sweeps_branching_and_smoothing(tiny):
    """The block protocol on a small population: temperatures are the rule applied to the residues BEFORE each block,
    the sweep counter advances by the block length, sum rules survive smoothing + branching."""
    o = _oracle_for(tiny); o.init_walkers(24)
    c0 = float(np.mean(o.chi2))
    T, ave, mn = o.anneal_selfcool(5, 4, n_boil=1, n_ramp=2, smooth_s=0.01)
    assert T[0] == 10.0 * c0 and ave[0] == c0 and o.sweep == 20
    for b in range(5):
        assert T[b] == oracle.selfcool_temperature(b, c0, ave[b], mn[b], 1, 2)
    wm = tiny.omega + 0.5 * tiny.domega
    np.testing.assert_allclose(o.a.sum(axis=1), tiny.A, rtol=1e-11)
    np.testing.assert_allclose((o.a * wm).sum(axis=1), tiny.B, rtol=1e-11)


def test_selfcool_block_is_smoothing_then_sweeps_then_branching(tiny):
    """"Once the transforms are smoothed and renormalized, they undergo Metropolis updates and branching.
    The process is then repeated."  One block of the protocol is therefore smooth -> k sweeps -> branch, in that order:
    replayed with the three public steps it gives the same state bit for bit, and the other order (sweeps -> smooth ->
    branch, the build's reading until round 2) does not."""
    W, k, s_amp, t = 24, 3, 0.05, 0.1
    o = _oracle_for(tiny); o.init_walkers(W)
    o.anneal(tiny.schedule[:4])                                      # a population that is not flat
    start_a, start_c, start_y, start_sweep = o.a.copy(), o.chi2.copy(), o.y.copy(), o.sweep

    def fresh():
        r = _oracle_for(tiny); r.init_walkers(W, start_a.copy())
        r.chi2[:] = start_c; r.y[:] = start_y; r.sweep = start_sweep
        return r

    p = fresh()
    T, _, _ = p.anneal_selfcool(1, k, n_boil=0, n_ramp=1, t_imprint=t, smooth_s=s_amp)
    a = fresh(); a.smooth(s_amp); a.anneal(np.full(k, T[0])); a.branch(T[0], t)
    b = fresh(); b.anneal(np.full(k, T[0])); b.smooth(s_amp); b.branch(T[0], t)
    np.testing.assert_array_equal(p.a, a.a)
    np.testing.assert_array_equal(p.chi2, a.chi2)
    assert not np.array_equal(p.a, b.a)


# ---- f2 branching fraction -----------------------------------------------------------
def test_branch_fraction_finds_the_temperature_that_kills_the_asked_fraction(tiny):
    """:174 'Delta is found numerically such that a given fraction of walkers is assigned a zero multiplier'.
    zeros(T) is 0 for T -> inf (all weights equal: every m = 1), grows as T falls, and the T found is the edge:
    zeros(T) >= n0 but a relative 1e-9 above it there are fewer."""
    o = _oracle_for(tiny); o.init_walkers(400)
    o.anneal(np.full(3, 1e5))
    assert o.branch_zeros(1e30) == 0
    zs = [o.branch_zeros(T) for T in np.std(o.chi2) * np.array([100.0, 10.0, 3.0, 1.0, 0.3, 0.1])]
    assert zs[0] <= zs[2] <= zs[4] and zs[-1] > zs[0]
    for frac in (0.25, 0.1, 0.5):
        n0 = int(np.floor(frac * o.W + 0.5))
        o2 = _oracle_for(tiny); o2.init_walkers(400, o.a.copy()); o2.chi2[:] = o.chi2; o2.sweep = o.sweep
        T, n_rec, mult, donor = o2.branch_fraction(frac, 0.1)
        assert T > 0 and mult.sum() == o.W and n_rec == (mult == 0).sum()
        assert n_rec >= n0 and n_rec - n0 <= 0.02 * o.W                      # the comb moves in small integer jumps
        assert o.branch_zeros(T) == n_rec and o.branch_zeros(T * (1 + 1e-9)) < n0
    flat = _oracle_for(tiny); flat.init_walkers(16)                           # identical walkers: nothing to branch
    assert flat.branch_fraction(0.25, 0.1)[0] == 0.0


# ---- f4 index selection by a truncated Markov walk -------------------------------------
def _selected_indices(o, a, n_moves, sweep=0):
    """p, s the oracle selects for moves 0..n_moves-1 of walker 0 on the FIXED spectrum a (T = 1e-300: nothing is
    ever accepted, so a never changes)."""
    ps = np.zeros((n_moves, 2), dtype=int)
    for m in range(n_moves):
        aa = a.copy(); M = np.zeros(o.P.n_tau); tr = o.move_raw(0, sweep, m, 1e-300, aa, M)
        ps[m] = tr["p"], tr["s"]
    return ps


def test_index_walk_limits_uniform_and_proportional_to_a(tiny):
    """:158 'If the walk has zero length, indices are selected randomly and uniformly ... In the limit of infinitely
    long walks, the indices are selected according to probability P(j) = a_j / A.'"""
    N = tiny.n_omega
    a = np.full(N, 1e-3); a[5] = 3.0; a[20] = 1.0; a[40] = 2.0            # three heavy bins: P = 1/2, 1/6, 1/3
    n = 3000
    o0 = _oracle_for(tiny, walk_len=0); o0.init_walkers(1)
    ps0 = _selected_indices(o0, a, n)
    assert (ps0[:, 0] != ps0[:, 1]).all()
    frac_heavy0 = np.isin(ps0[:, 0], [5, 20, 40]).mean()
    assert abs(frac_heavy0 - 3.0 / N) < 0.02                                # uniform: heavy bins are not preferred
    oL = _oracle_for(tiny, walk_len=1000); oL.init_walkers(1)     # ~47 proposals of a heavy bin per walk: mixed
    psL = _selected_indices(oL, a, n)
    assert (psL[:, 0] != psL[:, 1]).all()
    w = a / a.sum()
    for j in (5, 20, 40):
        assert abs((psL[:, 0] == j).mean() - w[j]) < 4 * np.sqrt(w[j] * (1 - w[j]) / n) + 0.01
    # s is drawn from the same law restricted to the bins other than p
    sel = psL[:, 0] == 5
    cond = a.copy(); cond[5] = 0.0; cond /= cond.sum()
    for j in (20, 40):
        assert abs((psL[sel, 1] == j).mean() - cond[j]) < 4 * np.sqrt(cond[j] * (1 - cond[j]) / sel.sum()) + 0.02


def test_index_walk_one_step_is_the_metropolis_rule_on_a(tiny):
    """One walk step by hand: from the uniform start j, the candidate c (Philox stream 2) replaces it iff u a_j < a_c."""
    N = tiny.n_omega
    rng = np.random.default_rng(7)
    a = rng.random(N) + 0.05
    o1 = _oracle_for(tiny, walk_len=1); o1.init_walkers(1)
    o0 = _oracle_for(tiny, walk_len=0); o0.init_walkers(1)
    ps1, ps0 = _selected_indices(o1, a, 200), _selected_indices(o0, a, 200)
    key = (o1.P.seed_lo, o1.P.seed_hi)
    moved = 0
    for m in range(200):
        x = oracle.philox4x32_10((0, 0, m, 2), key)
        x0 = oracle.philox4x32_10((0, 0, m, 0), key)
        p0 = (int(x0[0]) * N) >> 32
        c = (int(x[0]) * N) >> 32
        u = (int(x[1]) + 0.5) / 2.0 ** 32
        p1 = c if u * a[p0] < a[c] else p0
        assert ps0[m, 0] == p0 and ps1[m, 0] == p1
        moved += p1 != p0
    assert 20 < moved < 190


def test_index_walk_uniform_admixture(tiny):
    """:158 'a small fraction of the uniform distribution can be mixed in': with walk_uniform = f a fraction f of the
    moves keeps exactly the indices of the zero-length walk, the others exactly those of the pure walk."""
    N = tiny.n_omega
    a = np.random.default_rng(11).random(N) ** 4 + 1e-3
    n = 1500
    ps0 = _selected_indices(_mk(tiny, 0, 0.0), a, n)
    psw = _selected_indices(_mk(tiny, 5, 0.0), a, n)
    psm = _selected_indices(_mk(tiny, 5, 0.3), a, n)
    same_as_uniform = (psm == ps0).all(axis=1)
    same_as_walk = (psm == psw).all(axis=1)
    assert (same_as_uniform | same_as_walk).all()
    differs = ~(ps0 == psw).all(axis=1)
    frac = same_as_uniform[differs].mean()
    assert abs(frac - 0.3) < 4 * np.sqrt(0.3 * 0.7 / differs.sum())
    np.testing.assert_array_equal(_selected_indices(_mk(tiny, 5, 1.0), a, 200), ps0[:200])


def _mk(w, L, f):
    o = oracle.Oracle(w.omega, w.tau, w.F, w.sigma, w.A, w.B, w.eta, 1234, walk_len=L, walk_uniform=f)
    o.init_walkers(1)
    return o
