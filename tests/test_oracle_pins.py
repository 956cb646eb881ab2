"""Pins for the CPU oracle (oracle/rketd_oracle.cpp) — SURVEY.md §8(c) P1-P9.

The paper prints no field values (PAPER.md has no worked example; Figs. 2-3 are
absent), so every pin is a closed form, an invariant, a limiting case or brute
force, each chosen so that a plausible mistake in the oracle (dropped term, wrong
sign or index, transposed operand) fails at least one of them.  None of these
tests touches the CUDA path.
"""
import math
import os

import mpmath
import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

C0, MU0, EPS0 = oracle.constants()
ETA0 = math.sqrt(MU0 / EPS0)
DZ = 75e-6
DT = DZ / (2 * C0)


# ----------------------------------------------------------------------------- constants
def test_constants_are_si():
    assert C0 == 299792458.0
    assert MU0 == pytest.approx(4e-7 * math.pi, rel=1e-15)
    assert EPS0 * MU0 * C0 * C0 == pytest.approx(1.0, rel=1e-15)


# ----------------------------------------------------------------------------- G7: phi functions
@pytest.mark.parametrize("x", [0.0, 1e-300, 1e-13, 1.25e-4, 2.5e-3, 1.25e-2, 0.3, 0.49, 0.4999999, 0.5, 0.51, 1.0, 5.0, 40.0])
def test_phi_functions_against_50_digits(x):
    """phi1 = (1-e^-x)/x and phi2 = (e^-x-1+x)/x^2 — the brackets of eq. (11)."""
    mpmath.mp.dps = 50 if x == 0.0 or x > 1e-10 else int(50 - 2 * math.log10(x))   # 1 - e^-x needs the digits
    p1, p2 = oracle.phi(x)
    if x == 0.0:
        assert (p1, p2) == (1.0, 0.5)
        return
    xm = mpmath.mpf(x)
    r1 = (1 - mpmath.exp(-xm)) / xm
    r2 = (mpmath.exp(-xm) - 1 + xm) / xm ** 2
    assert abs(p1 - r1) / r1 < 3e-16
    assert abs(p2 - r2) / r2 < 4.5e-16


def test_coefficients_vacuum_and_limits():
    """Vacuum: ca = 1, ch = dt/(eps0 dz), kb = kc = 0, ka = e^{-nu dt}; chh = dt/(mu0 dz); Mur m."""
    wp = np.array([0.0, 0.0, 2 * math.pi * 28.7e9])
    nu = np.array([0.0, 2e10, 0.0])
    c = oracle.coefficients(wp, nu, DZ, DT)
    assert c["ca"][0] == 1.0 and c["ca"][1] == 1.0
    assert c["ch"][0] == pytest.approx(DT / (EPS0 * DZ), rel=1e-15)
    assert c["kb"][0] == 0.0 and c["kc"][0] == 0.0 and c["kb"][1] == 0.0
    assert c["ka"][0] == 1.0 and c["ka"][1] == pytest.approx(math.exp(-2e10 * DT), rel=1e-15)
    assert c["chh"] == pytest.approx(DT / (MU0 * DZ), rel=1e-15)
    assert c["m"] == pytest.approx(-1.0 / 3.0, rel=1e-12)          # S = 0.5
    assert oracle.coefficients(wp, nu, DZ, DZ / C0)["m"] == pytest.approx(0.0, abs=1e-15)   # S = 1
    # nu = 0 plasma: (11) becomes the trapezoid rule J' = J + eps0 wp^2 (dt/2)(E' + E)
    w2 = wp[2] ** 2
    assert c["ka"][2] == 1.0
    assert c["kb"][2] == pytest.approx(EPS0 * w2 * DT / 2, rel=1e-14)
    assert c["kc"][2] == pytest.approx(EPS0 * w2 * DT / 2, rel=1e-14)


def test_coefficients_against_50_digit_closed_form():
    """ca, cj, ch, ka, kb, kc from eliminating J^{n+1} between eqs. (11) and (12), in 50 digits."""
    mpmath.mp.dps = 50
    rng = np.random.default_rng(7)
    wp = rng.uniform(2 * math.pi * 5e9, 2 * math.pi * 60e9, 40)
    nu = np.concatenate([rng.uniform(0, 1e11, 30), [1e-3, 1e3, 1e6, 1e9, 4e12, 8e12, 1e13, 5e13, 1.0, 1e11]])
    c = oracle.coefficients(wp, nu, DZ, DT)
    dt, dz, e0 = mpmath.mpf(DT), mpmath.mpf(DZ), 1 / (mpmath.mpf(MU0) * mpmath.mpf(C0) ** 2)
    for i in range(40):
        w, v = mpmath.mpf(wp[i]), mpmath.mpf(nu[i])
        a = mpmath.exp(-v * dt)
        b11 = (1 - a) / v * e0 * w ** 2                      # coefficient of E^n in (11), first bracket
        c11 = (a - 1 + v * dt) / (v ** 2 * dt) * e0 * w ** 2   # coefficient of (E^{n+1} - E^n) in (11)
        D = 1 + dt / (2 * e0) * c11
        ref = {"ca": (1 - dt / (2 * e0) * (b11 - c11)) / D, "cj": dt / (2 * e0) * (1 + a) / D,
               "ch": dt / (e0 * dz) / D, "ka": a, "kb": b11 - c11, "kc": c11}
        for k, r in ref.items():
            # eps0 itself is a rounded double in the oracle: allow a few ulp; kb = b - c is a
            # difference of two rounded numbers of similar size (b ~ 2c for small x), a few ulp more
            assert abs(c[k][i] - r) <= (5e-15 if k == "kb" else 8e-16) * abs(r), (k, i, c[k][i], r)


# ----------------------------------------------------------------------------- P1
def test_P1_courant_one_translation_and_exact_mur():
    """wp = 0, S = 1: a right-going pulse moves exactly one cell per step; Mur (m = 0) absorbs it exactly."""
    N, n1 = 400, 150
    dt = DZ / C0
    k = np.arange(N, dtype=np.float64)
    f = lambda s: np.exp(-((s - 120.0) / 12.0) ** 2) * np.sin(0.3 * s)
    st = oracle.State(N, 1, E0=f(k), H0=f(k + 1.0) / ETA0)
    z = np.zeros((1, N))
    oracle.run(st, z, z, DZ, dt, n1)
    expect = f(k - n1)
    assert np.max(np.abs(st.E[0] - expect)) < 5e-14      # rounding of S = 1 only; a wrong index gives O(1)
    # left-going pulse: H = -E/eta0 at the mirrored stagger; translates the other way
    st = oracle.State(N, 1, E0=f(k), H0=-f(k) / ETA0)
    oracle.run(st, z, z, DZ, dt, 60)
    assert np.max(np.abs(st.E[0] - f(k + 60))) < 5e-14
    # run the right-going pulse out through the right boundary: nothing comes back
    st = oracle.State(N, 1, E0=f(k), H0=f(k + 1.0) / ETA0)
    oracle.run(st, z, z, DZ, dt, 500)
    assert np.max(np.abs(st.E[0])) < 1e-13


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("nu", [2.4e12, 8e12])     # x = 0.30 (series branch) and 1.0 (formula branch)
def test_P2_residual_of_literal_eq11_and_eq12(nu):
    """After each step the state satisfies eq. (12) and eq. (11) as PRINTED."""
    N = 64
    rng = np.random.default_rng(3)
    wp = np.full((1, N), 2 * math.pi * 40e9)
    nuv = np.full((1, N), nu)
    st = oracle.State(N, 1, E0=rng.uniform(-1, 1, N), H0=rng.uniform(-1, 1, N) / ETA0, J0=rng.uniform(-1, 1, N) * 1e3)
    a = math.exp(-nu * DT)
    for _ in range(20):
        E0, J0 = st.E[0].copy(), st.J[0].copy()
        oracle.run(st, wp, nuv, DZ, DT, 1)
        E1, J1, H = st.E[0], st.J[0], st.H[0]
        w2 = wp[0] ** 2
        j11 = a * J0 + (1 - a) / nu * EPS0 * w2 * E0 + (a - 1 + nu * DT) / (nu ** 2 * DT) * (EPS0 * w2 * E1 - EPS0 * w2 * E0)
        assert np.max(np.abs(J1 - j11)) <= 1e-12 * np.max(np.abs(J1))
        k = np.arange(1, N - 1)
        e12 = E0[k] - DT / (EPS0 * DZ) * (H[k] - H[k - 1]) - DT / (2 * EPS0) * (J1[k] + J0[k])
        assert np.max(np.abs(E1[k] - e12)) <= 1e-12 * np.max(np.abs(E1))


def test_P2_H_update_is_eq14():
    N = 32
    rng = np.random.default_rng(5)
    E0, H0 = rng.uniform(-1, 1, N), rng.uniform(-1, 1, N)
    H0[N - 1] = 0.0
    st = oracle.State(N, 1, E0=E0, H0=H0)
    z = np.zeros((1, N))
    oracle.run(st, z, z, DZ, DT, 1)
    k = np.arange(N - 1)
    assert np.allclose(st.H[0][k], H0[k] - DT / (MU0 * DZ) * (E0[k + 1] - E0[k]), rtol=0, atol=1e-18)
    assert st.H[0][N - 1] == 0.0


# ----------------------------------------------------------------------------- P3
def _energy(E, Hnew, Hold, J, wp):
    w = EPS0 * np.sum(E ** 2) + MU0 * np.sum(Hnew[:-1] * Hold[:-1])
    pl = wp > 0
    return 0.5 * DZ * (w + np.sum(J[pl] ** 2 / (EPS0 * wp[pl] ** 2)))


@pytest.mark.parametrize("case", ["vacuum", "lossless_slab", "lossy_slab"])
def test_P3_discrete_energy(case):
    """W^n = eps0 sum E^2 + mu0 sum H^{n+1/2} H^{n-1/2} + sum J^2/(eps0 wp^2): conserved when nu = 0."""
    N, nsteps = 600, 3000
    wp = np.zeros((1, N))
    nu = np.zeros((1, N))
    if case != "vacuum":
        wp[0, 250:370] = 2 * math.pi * 28.7e9
    if case == "lossy_slab":
        nu[0, 250:370] = 2e10
    k = np.arange(N, dtype=np.float64)
    E0 = np.exp(-((k - 120.0) / 15.0) ** 2)
    E0[0] = E0[-1] = 0.0
    # start from E^0 and H^{-1/2}: take one oracle step first so that both H half-levels are at hand
    st = oracle.State(N, 1, E0=E0)
    W = []
    Hold = st.H[0].copy()
    for n in range(nsteps):
        # energy at integer step n needs H^{n+1/2} (after this step's H update) and H^{n-1/2} (before)
        E_n, J_n = st.E[0].copy(), st.J[0].copy()
        oracle.run(st, wp, nu, DZ, DT, 1, boundary=oracle.BOUNDARY_PEC)
        Hnew = st.H[0].copy()
        W.append(_energy(E_n, Hnew, Hold, J_n, wp[0]))
        Hold = Hnew
    W = np.array(W)
    if case == "lossy_slab":
        assert np.all(np.diff(W) <= 1e-13 * W[0])
        assert W[-1] < 0.9 * W[0]
    else:
        # printed eq. (13) (without 1/D on the J and curl terms) drifts by ~3e-5 here
        assert np.max(np.abs(W / W[0] - 1.0)) < 2e-13


# ----------------------------------------------------------------------------- P4
@pytest.mark.parametrize("nu", [0.0, 1e6, 2e10, 1e11])
def test_P4_J_is_exact_solution_of_eq6_for_piecewise_linear_E(nu):
    """Brute force: RK4 (64 sub-steps per dt) of dJ/dt + nu J = eps0 wp^2 E(t), E linear on each step."""
    N, nsteps, cell = 200, 400, 100
    wpv = 2 * math.pi * 28.7e9
    wp = np.zeros((1, N)); nuv = np.zeros((1, N))
    wp[0, 80:130] = wpv; nuv[0, 80:130] = nu
    st = oracle.State(N, 1)
    rec, recJ = oracle.run(st, wp, nuv, DZ, DT, nsteps, src_kind=0, src_params=(20e-12, 80e-12, 1.0),
                           src_cell=40, probes=[cell], record_J=True)
    Es = np.concatenate([[0.0], rec[0, 0]])
    Js = np.concatenate([[0.0], recJ[0, 0]])
    assert np.max(np.abs(Js)) > 0
    nsub = 64
    h = DT / nsub
    J = 0.0
    Jref = [0.0]
    for n in range(nsteps):
        e0, e1 = Es[n], Es[n + 1]
        f = lambda t, j: -nu * j + EPS0 * wpv ** 2 * (e0 + (e1 - e0) * t / DT)
        for s in range(nsub):
            t = s * h
            k1 = f(t, J); k2 = f(t + h / 2, J + h / 2 * k1); k3 = f(t + h / 2, J + h / 2 * k2); k4 = f(t + h, J + h * k3)
            J += h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        Jref.append(J)
    Jref = np.array(Jref)
    assert np.max(np.abs(Js - Jref)) < 5e-13 * np.max(np.abs(Jref))
    if nu == 0.0:
        trap = np.concatenate([[0.0], np.cumsum(EPS0 * wpv ** 2 * DT / 2 * (Es[1:] + Es[:-1]))])
        assert np.max(np.abs(Js - trap)) < 1e-13 * np.max(np.abs(trap))


# ----------------------------------------------------------------------------- P5
def _slab_rt_analytic(f, wp, nu, d):
    """Single homogeneous Drude slab in vacuum, normal incidence, e^{+jwt} convention."""
    w = 2 * np.pi * f
    eps = 1 - wp ** 2 / (w ** 2 - 1j * w * nu)
    n = np.sqrt(eps)
    n = np.where(n.imag > 0, -n, n)
    k = n * w / C0
    r = (1 - n) / (1 + n)
    P = np.exp(-2j * k * d)
    R = r * (1 - P) / (1 - r ** 2 * P)
    T = (1 - r ** 2) * np.exp(-1j * k * d) / (1 - r ** 2 * P)
    return np.abs(R), np.abs(T)


def test_P5_slab_reflection_transmission_matches_analytic():
    """Config 1 (PAPER.md:123-132 at 1/10 thickness): |R|, |T| from FFTs of probe records vs transfer matrix."""
    w = wl.config1()
    tot = oracle.run_workload(w)["rec"][0]
    # vacuum reference run: same source, same probes, same initial noise, no slab
    wv = wl.config1()
    wv.media = lambda lo=0, hi=w.ncells, b0=0, b1=1: (np.zeros((b1 - b0, hi - lo)), np.zeros((b1 - b0, hi - lo)))
    inc = oracle.run_workload(wv)["rec"][0]
    F = lambda x: np.fft.rfft(x)
    freqs = np.fft.rfftfreq(w.nsteps, w.dt)
    Iinc_r, Iinc_t = F(inc[0]), F(inc[1])
    R = np.abs(F(tot[0] - inc[0])) / np.abs(Iinc_r)
    T = np.abs(F(tot[1])) / np.abs(Iinc_t)
    band = np.abs(Iinc_r) >= 1e-2 * np.max(np.abs(Iinc_r))
    assert 15 <= band.sum() <= 30 and freqs[band].min() < 2e9 and freqs[band].max() > 25e9
    Ra, Ta = _slab_rt_analytic(freqs[band], 2 * math.pi * 28.7e9, 2.0e10, 120 * w.dz)
    assert np.max(np.abs(R[band] - Ra)) < 1e-2
    assert np.max(np.abs(T[band] - Ta)) < 1e-2
    # the analytic side itself is held by a stored table (tests/golden/slab_rt_analytic.txt)
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "slab_rt_analytic.txt"))
    Rg, Tg = _slab_rt_analytic(gold[:, 0] * 1e9, 2 * math.pi * 28.7e9, 2.0e10, 9e-3)
    assert np.max(np.abs(Rg - gold[:, 1])) < 2e-6 and np.max(np.abs(Tg - gold[:, 2])) < 2e-6


# ----------------------------------------------------------------------------- P6
@pytest.mark.parametrize("fp,nu", [(60e9, 0.0), (60e9, 1e11), (5e9, 0.0), (40e9, 1e9), (60e9, 1e3), (60e9, 1e-3)])
def test_P6_stability(fp, nu):
    N = 256
    rng = np.random.default_rng(11)
    st = oracle.State(N, 1, E0=rng.uniform(-1, 1, N))
    st.E[0, 0] = st.E[0, -1] = 0.0
    wp = np.full((1, N), 2 * math.pi * fp)
    oracle.run(st, wp, np.full((1, N), nu), DZ, DT, 20000, boundary=oracle.BOUNDARY_PEC)
    assert np.max(np.abs(st.E)) <= 2.0 and np.all(np.isfinite(st.J))


# ----------------------------------------------------------------------------- P7
def test_P7_domain_of_dependence_window_is_bit_exact():
    w = wl.config4(ncells=40_000, nsteps=300)
    w.probes = np.array([10_000, 20_000, 31_234], np.int64)
    full = oracle.run_workload(w)["rec"][0]
    for i, p in enumerate(w.probes):
        win = oracle.run_workload(w, cells=(int(p) - 301, int(p) + 302))
        assert win["probe_cells"] == [int(p)]
        assert np.array_equal(win["rec"][0][0], full[i])
    # and one step too few of margin is visible: the window really is the light cone
    p = int(w.probes[0])
    short = oracle.run_workload(w, cells=(p - 150, p + 151))["rec"][0][0]
    assert not np.array_equal(short, full[0]) and np.array_equal(short[:150], full[0][:150])


# ----------------------------------------------------------------------------- P8
def test_P8_running_dft_equals_direct_dft():
    w = wl.config5(nbatch=3, nsteps=700)
    out = oracle.run_workload(w)
    w2 = wl.config5(nbatch=3, nsteps=700, dft=False)
    rec = oracle.run_workload(w2)["rec"]
    n = np.arange(1, 701)
    tw = np.exp(-2j * np.pi * w.dft_freqs[:, None] * (n[None, :] * w.dt))
    X = np.einsum("bpn,fn->bpf", rec, tw)
    assert out["dft_mag"].shape == (3, 2, 64)
    assert np.max(np.abs(out["dft_mag"] - np.abs(X))) < 1e-13 * np.max(np.abs(X))
    assert np.max(np.abs(X)) > 1.0


# ----------------------------------------------------------------------------- P9
def test_P9_openmp_build_is_bit_identical():
    for w in (wl.config1(nsteps=800), wl.config3(ncells=512, nbatch=9, nsteps=300)):
        a = oracle.run_workload(w, omp=False)
        b = oracle.run_workload(w, omp=True)
        assert np.array_equal(a["rec"], b["rec"])
        assert np.array_equal(a["state"].J, b["state"].J) and np.array_equal(a["state"].H, b["state"].H)


# ----------------------------------------------------------------------------- source, continuation
def test_source_waveform_eq15_unit_peak():
    tau, t0 = 20e-12, 80e-12
    n = np.arange(0, 2000)
    s = np.array([oracle.source(0, (tau, t0, 1.0), int(i), DT) for i in n])
    t = (n + 1) * DT
    ref = (t - t0) / tau * np.exp(0.5 - (t - t0) ** 2 / (2 * tau ** 2))
    assert np.max(np.abs(s - ref)) < 1e-15
    assert abs(np.max(s) - 1.0) < 1e-4 and abs(np.min(s) + 1.0) < 1e-4      # unit peak (at t0 +- tau)
    assert oracle.source(1, (3.0, 4.0, 5.0), 1, DT) == 4.0 and oracle.source(1, (3.0,), 7, DT) == 0.0


def test_run_is_restartable():
    w = wl.config1(nsteps=500)
    a = oracle.run_workload(w)
    wp, nu = w.media_full()
    st = oracle.State(w.ncells, 1, w.initial_E_full())
    parts = []
    for n in (1, 199, 300):
        r, _ = oracle.run(st, wp, nu, w.dz, w.dt, n, src_kind=w.src_kind, src_params=w.src_params,
                          src_cell=w.src_cell, probes=w.probes)
        parts.append(r)
    assert np.array_equal(np.concatenate(parts, axis=2), a["rec"])
    assert np.array_equal(st.E, a["state"].E)


def test_soft_source_and_probe_timing():
    """One step from rest: E'[ks] = s[1] exactly, everything else 0; sample 0 is time dt (a4, a6, G12, G14)."""
    N = 50
    st = oracle.State(N, 1)
    z = np.zeros((1, N))
    rec, _ = oracle.run(st, z, z, DZ, DT, 3, src_kind=1, src_params=(0.25, 0.0, 0.0), src_cell=20, probes=[20, 21, 19])
    assert rec[0, 0, 0] == 0.25 and rec[0, 1, 0] == 0.0
    # vacuum, S = 1/2: E'[k+-1] = S^2 * E[k] after one more step
    assert rec[0, 1, 1] == pytest.approx(0.25 * 0.25, rel=1e-14) and rec[0, 2, 1] == pytest.approx(0.0625, rel=1e-14)
    assert rec[0, 0, 1] == pytest.approx(0.25 * (1 - 2 * 0.25), rel=1e-14)


def test_mur_reflection_is_small_at_half_courant():
    """Mur-1 at S = 1/2 is not exact, but a well-resolved pulse leaves < 1e-3 behind."""
    N = 800
    k = np.arange(N, dtype=np.float64)
    f = lambda s: np.exp(-((s - 500.0) / 40.0) ** 2)
    st = oracle.State(N, 1, E0=f(k), H0=f(k + 0.75) / ETA0)     # right-going at S = 1/2: H at (k+1/2) dz, t = -dt/2
    z = np.zeros((1, N))
    oracle.run(st, z, z, DZ, DT, 2000)
    assert np.max(np.abs(st.E)) < 1e-3


# ----------------------------------------------------------------------------- paper experiment A (NEXT-1)
def test_paper_experiment_A_reflection_transmission():
    """The paper's own experiment (Figs. 2-3): 4096 cells, 9 cm slab (1200 cells), dt = 125 fs,
    tau = 15 dt.  |R|, |T| by FFT against the closed form.  T holds to 1e-3 over the whole pulse band
    (1-300 GHz); R to 1e-2 up to 150 GHz and 2e-2 above, where the line has < 27 cells per wavelength and the
    first-order Mur end reflects about 1 % (the paper used PML there)."""
    w = wl.paper_exp_a()
    assert w.ncells == 4096 and w.slab == (1448, 1200) and abs(w.src_params[0] - 15 * 125e-15) < 1e-25
    tot = oracle.run_workload(w)["rec"][0]
    wv = wl.paper_exp_a()
    wv.media = lambda lo=0, hi=w.ncells, b0=0, b1=1: (np.zeros((b1 - b0, hi - lo)), np.zeros((b1 - b0, hi - lo)))
    inc = oracle.run_workload(wv)["rec"][0]
    assert np.max(np.abs(tot[:, -200:])) < 1e-5 * np.max(np.abs(tot))          # records have decayed
    freqs = np.fft.rfftfreq(w.nsteps, w.dt)
    Ir, It = np.fft.rfft(inc[0]), np.fft.rfft(inc[1])
    R = np.abs(np.fft.rfft(tot[0] - inc[0])) / np.abs(Ir)
    T = np.abs(np.fft.rfft(tot[1])) / np.abs(It)
    band = np.abs(Ir) >= 1e-2 * np.max(np.abs(Ir))
    assert freqs[band].min() < 2e9 and freqs[band].max() > 250e9
    Ra, Ta = _slab_rt_analytic(freqs[band], 2 * math.pi * 28.7e9, 2.0e10, 1200 * w.dz)
    low = freqs[band] <= 150e9
    assert np.max(np.abs(T[band] - Ta)) < 1e-3
    assert np.max(np.abs(R[band][low] - Ra[low])) < 1e-2
    assert np.max(np.abs(R[band] - Ra)) < 2e-2
    # opaque below the plasma frequency, transparent far above it
    assert T[band][freqs[band] < 25e9].max() < 1e-5 and T[band][freqs[band] > 200e9].min() > 0.9


# ----------------------------------------------------------------------------- first-order ETD, eq. (9) (NEXT-4)
@pytest.mark.parametrize("nu", [2.4e12, 8e12, 2e10])
def test_ETD1_residual_of_literal_eq9_and_eq12(nu):
    """scheme 1: after each step the state satisfies eq. (9) and eq. (12) as PRINTED."""
    N = 64
    rng = np.random.default_rng(4)
    wp = np.full((1, N), 2 * math.pi * 40e9)
    nuv = np.full((1, N), nu)
    st = oracle.State(N, 1, E0=rng.uniform(-1, 1, N), H0=rng.uniform(-1, 1, N) / ETA0, J0=rng.uniform(-1, 1, N) * 1e3)
    a = math.exp(-nu * DT)
    for _ in range(20):
        E0, J0 = st.E[0].copy(), st.J[0].copy()
        oracle.run(st, wp, nuv, DZ, DT, 1, scheme=oracle.SCHEME_ETD1)
        E1, J1, H = st.E[0], st.J[0], st.H[0]
        Fn = EPS0 * wp[0] ** 2 * E0
        j9 = J0 * a - Fn * (a - 1) / nu                                   # eq. (9) as printed
        assert np.max(np.abs(J1 - j9)) <= 1e-11 * np.max(np.abs(J1))       # (a - 1)/nu cancels 3 digits at nu = 2e10
        k = np.arange(1, N - 1)
        e12 = E0[k] - DT / (EPS0 * DZ) * (H[k] - H[k - 1]) - DT / (2 * EPS0) * (J1[k] + J0[k])
        assert np.max(np.abs(E1[k] - e12)) <= 1e-12 * np.max(np.abs(E1))


@pytest.mark.parametrize("nu", [0.0, 2e10, 1e11])
def test_ETD1_J_is_exact_solution_of_eq6_for_piecewise_constant_E(nu):
    """Brute force for eq. (9): RK4 (64 sub-steps per dt) of dJ/dt + nu J = eps0 wp^2 E^n, E HELD at its value at
    the start of each step (eq. (8): F = F_n) reproduces the scheme-1 J series; and the two schemes differ at first
    order in dt (they are not the same recurrence)."""
    N, nsteps, cell = 200, 400, 100
    wpv = 2 * math.pi * 28.7e9
    wp = np.zeros((1, N)); nuv = np.zeros((1, N))
    wp[0, 80:130] = wpv; nuv[0, 80:130] = nu
    kw = dict(src_kind=0, src_params=(20e-12, 80e-12, 1.0), src_cell=40, probes=[cell], record_J=True)
    rec, recJ = oracle.run(oracle.State(N, 1), wp, nuv, DZ, DT, nsteps, scheme=oracle.SCHEME_ETD1, **kw)
    Es = np.concatenate([[0.0], rec[0, 0]])
    Js = np.concatenate([[0.0], recJ[0, 0]])
    nsub, J, Jref = 64, 0.0, [0.0]
    h = DT / nsub
    for n in range(nsteps):
        f = lambda j: -nu * j + EPS0 * wpv ** 2 * Es[n]
        for s in range(nsub):
            k1 = f(J); k2 = f(J + h / 2 * k1); k3 = f(J + h / 2 * k2); k4 = f(J + h * k3)
            J += h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        Jref.append(J)
    Jref = np.array(Jref)
    assert np.max(np.abs(Jref)) > 0 and np.max(np.abs(Js - Jref)) < 5e-13 * np.max(np.abs(Jref))
    rec2, _ = oracle.run(oracle.State(N, 1), wp, nuv, DZ, DT, nsteps, **kw)
    d = np.max(np.abs(rec2 - rec)) / np.max(np.abs(rec2))
    assert 1e-5 < d < 5e-2, d


def test_ETD1_coefficients_closed_form_and_vacuum():
    wp = np.array([0.0, 2 * math.pi * 28.7e9, 2 * math.pi * 60e9])
    nu = np.array([0.0, 2e10, 0.0])
    c = oracle.coefficients(wp, nu, DZ, DT, oracle.SCHEME_ETD1)
    mpmath.mp.dps = 50
    for i in range(3):
        x = mpmath.mpf(nu[i]) * mpmath.mpf(DT)
        a = mpmath.exp(-x)
        beta = mpmath.mpf(DT) if nu[i] == 0 else (1 - a) / mpmath.mpf(nu[i])
        w2 = mpmath.mpf(wp[i]) ** 2
        ref = {"ca": 1 - w2 * beta * mpmath.mpf(DT) / 2, "cj": mpmath.mpf(DT) / (2 * mpmath.mpf(EPS0)) * (1 + a),
               "ch": mpmath.mpf(DT) / (mpmath.mpf(EPS0) * mpmath.mpf(DZ)), "ka": a, "kb": mpmath.mpf(EPS0) * w2 * beta,
               "kc": mpmath.mpf(0)}
        for k, v in ref.items():
            assert abs(c[k][i] - float(v)) <= 4e-16 * abs(float(v)), (k, i)


# ----------------------------------------------------------------------------- PML (NEXT-2)
def _end_reflection(boundary, pml=(0, 0.0, 1.0), tau=20e-12, N=2000):
    """Peak of what comes back from the left end / peak of what went in, seen at node 600 (source at node 1000)."""
    z = np.zeros((1, N))
    st = oracle.State(N, 1)
    tc = int(4 * tau / DT)
    rec, _ = oracle.run(st, z, z, DZ, DT, tc + 4400, src_kind=0, src_params=(tau, 4 * tau, 1.0), src_cell=1000,
                        probes=[600], boundary=boundary, pml=pml)
    r = rec[0, 0]
    cut = tc + 2000                      # incident passes by step tc + 800, the echo arrives at step tc + 3200
    return np.abs(r[cut:]).max() / np.abs(r[:cut]).max()


def test_PML_with_R0_1_is_the_PEC_run_bit_for_bit():
    """sigma = 0 (R0 = 1): the layer is vacuum and the run must equal the PEC-terminated one bit for bit (indexing of
    the layer, of the mirrored right end and of the conductor behind it)."""
    w = wl.config1(nsteps=3000)
    a = oracle.run_workload(w, boundary=oracle.BOUNDARY_PEC)
    b = oracle.run_workload(w, boundary=oracle.BOUNDARY_PML, pml=(5, 3.0, 1.0))
    assert np.array_equal(a["rec"], b["rec"]) and np.array_equal(a["state"].H, b["state"].H)
    assert _end_reflection(oracle.BOUNDARY_PEC) > 0.99


def test_PML_matched_layer_attenuates_by_R0_per_round_trip():
    """Constant profile (m = 0): a matched lossy medium is dispersion-free, a pulse keeps its shape and decays as
    exp(-sigma eta0 x) = R0^(x / 2d).  Pins sigma_max, the matching sigma* = sigma mu0/eps0 and the signs."""
    N, npml, R0 = 1400, 600, 1e-3
    z = np.zeros((1, N))
    st = oracle.State(N, 1)
    probes = [500, 400, 300]                           # 100, 200, 300 nodes inside the left layer (interface at 600)
    rec, _ = oracle.run(st, z, z, DZ, DT, 1800, src_kind=0, src_params=(20e-12, 80e-12, 1.0), src_cell=700,
                        probes=probes, boundary=oracle.BOUNDARY_PML, pml=(npml, 0.0, R0))
    pk = np.abs(rec[0]).max(1)
    want = R0 ** (100.0 / (2 * npml))
    assert abs(pk[1] / pk[0] - want) < 2e-3 * want and abs(pk[2] / pk[1] - want) < 2e-3 * want


def test_PML_reflection_floor_against_Mur():
    """What the paper's 5-cell layer buys (reading: cubic grading, R0 = 1e-6).  For the paper's own pulse
    (tau = 15 dt, content to 300 GHz) it reflects 7 x less than first-order Mur at S = 1/2, 10 cells 30 x less;
    for the slow BASELINE pulse (tau = 20 ps) first-order Mur is already at 5e-5 and the 5-cell layer is not better."""
    tau_paper = 15 * 125e-15
    mur, pml5, pml10 = (_end_reflection(oracle.BOUNDARY_MUR, tau=tau_paper),
                        _end_reflection(oracle.BOUNDARY_PML, (5, 3.0, 1e-6), tau=tau_paper),
                        _end_reflection(oracle.BOUNDARY_PML, (10, 3.0, 1e-6), tau=tau_paper))
    assert 1e-3 < mur < 3e-3 and pml5 < mur / 5 and pml10 < mur / 25
    assert _end_reflection(oracle.BOUNDARY_MUR) < 1e-4 and _end_reflection(oracle.BOUNDARY_PML, (5, 3.0, 1e-6)) < 1e-3


def test_PML_is_mirror_symmetric():
    """Source on the centre node of an odd grid: E is even about it, so mirrored probes record the same series
    (the right layer's H index N-2-j and E index N-1-j)."""
    N = 401
    z = np.zeros((1, N))
    rec, _ = oracle.run(oracle.State(N, 1), z, z, DZ, DT, 1500, src_kind=0, src_params=(1.875e-12, 7.5e-12, 1.0), src_cell=200,
                        probes=[2, 398, 0, 400, 4, 396], boundary=oracle.BOUNDARY_PML, pml=(5, 3.0, 1e-6))
    r = rec[0]
    assert np.abs(r[0]).max() > 1e-4
    assert np.array_equal(r[0], r[1]) and np.array_equal(r[4], r[5]) and not r[2].any() and not r[3].any()


# ----------------------------------------------------------------------------- R/T sweep from DFT accumulators (NEXT-4)
def test_sweep_RT_from_running_dft_matches_analytic():
    """Config-3 slabs (12 grids: drawn thickness, wp, nu): |R|, |T| from the oracle's running DFT (row a7) of a slab
    run and of one vacuum run, against the closed form.  Pins the DFT sign/phase convention (a wrong sign of the
    exponent or an off-by-one in the sample time would not cancel in X_slab - X_vac)."""
    nb, freqs = 12, np.linspace(2e9, 26e9, 13)
    w = wl.config3(nbatch=nb)
    w.dft_freqs = freqs
    wv = wl.config3(nbatch=1)
    wv.dft_freqs = freqs
    wv.media = lambda lo=0, hi=w.ncells, b0=0, b1=1: (np.zeros((b1 - b0, hi - lo)), np.zeros((b1 - b0, hi - lo)))
    X = oracle.run_workload(w, omp=True)["dft"]
    inc = oracle.run_workload(wv)["dft"][0]
    R = np.abs(X[:, 0] - inc[0]) / np.abs(inc[0])
    T = np.abs(X[:, 1]) / np.abs(inc[1])
    wp, nu = w.media(2000, 2001, 0, nb)
    thick = (w.media(0, w.ncells, 0, nb)[0] > 0).sum(1)
    for g in range(nb):
        Ra, Ta = _slab_rt_analytic(freqs, wp[g, 0], nu[g, 0], thick[g] * w.dz)
        assert np.abs(R[g] - Ra).max() < 1e-3 and np.abs(T[g] - Ta).max() < 1e-3, g
