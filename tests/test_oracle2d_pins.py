"""Pins for the 2-D TMz half of the CPU oracle (oracle/rketd_oracle.cpp, oracle2d_*) — SURVEY §8(f) NEXT-3.

The paper gives the vector equations (1)-(3) and names the 2-D generalisation as its next step
 but prints nothing 2-D.  What fixes the 2-D oracle is therefore: its reduction to the (pinned) 1-D
oracle when the fields do not vary along one axis (Q1, both axes), the energy invariant of the lossless leapfrog in
a conducting box (Q2), the eigenmodes of that box, which follow the Yee dispersion relation exactly (Q3, with
dx != dy so that an exchanged step or coefficient shows), the exact solution of eq. (6) for the current (Q4),
the symmetry under exchange of the axes (Q5), the domain of dependence (Q7) and OpenMP == serial (Q8).
None of these tests touches the CUDA path.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1709_00821_b200 import workloads as wl

C0, MU0, EPS0 = oracle.constants()
DX = 75e-6
DT = DX / (2 * C0)
SRC = (20e-12, 80e-12, 1.0)


def _slab_media_1d(n, lo, hi, wp0=2 * math.pi * 28.7e9, nu0=2e10):
    wp = np.zeros(n); nu = np.zeros(n)
    wp[lo:hi] = wp0; nu[lo:hi] = nu0
    return wp, nu


# ----------------------------------------------------------------------------- Q1
@pytest.mark.parametrize("axis", ["x", "y"])
def test_Q1_uniform_along_one_axis_is_the_1d_oracle_bit_for_bit(axis):
    """Fields and media that do not vary along one axis stay so (away from that axis' edges: a disturbance travels at
    most one node per step), the differences along it vanish exactly, and what is left is eqs. (11), (12), (14) of
    the 1-D method with Mur at the two ends: Ez <-> Ex, Hy <-> -H (variation along x) or Hx <-> +H (along y)."""
    n, nother, nsteps = 300, 2 * 120 + 9, 110          # nsteps < (nother - 1)/2: the middle line is untouched
    dvar, doth = DX, 1.7 * DX                           # different steps: the step of the uniform axis must not matter
    wp1, nu1 = _slab_media_1d(n, 140, 190)
    k = np.arange(n, dtype=np.float64)
    E1 = np.exp(-((k - 100.0) / 12.0) ** 2)
    rng = np.random.default_rng(5)
    H1 = 1e-3 * rng.uniform(-1, 1, n); H1[-1] = 0.0
    J1 = 1e-2 * rng.uniform(-1, 1, n) * (wp1 > 0)
    st1 = oracle.State(n, 1, E0=E1, H0=H1, J0=J1)
    probes1 = [0, 1, 60, 150, 189, n - 2, n - 1]
    rec1, _ = oracle.run(st1, wp1[None], nu1[None], dvar, DT, nsteps, probes=probes1)
    mid = nother // 2
    if axis == "x":    # variation along x: arrays [ny = nother][nx = n]
        rep = lambda a: np.repeat(a[None, :], nother, 0)
        st2 = oracle.State2D(n, nother, Ez0=rep(E1), Hy0=rep(-H1), Jz0=rep(J1))
        rec2, _ = oracle.run2d(st2, rep(wp1), rep(nu1), dvar, doth, DT, nsteps, probes=[(p, mid) for p in probes1])
        E2, Hvar, Hoth, J2 = st2.Ez[mid], -st2.Hy[mid], st2.Hx[mid], st2.Jz[mid]
    else:              # variation along y: arrays [ny = n][nx = nother]
        rep = lambda a: np.repeat(a[:, None], nother, 1)
        st2 = oracle.State2D(nother, n, Ez0=rep(E1), Hx0=rep(H1), Jz0=rep(J1))
        rec2, _ = oracle.run2d(st2, rep(wp1), rep(nu1), doth, dvar, DT, nsteps, probes=[(mid, p) for p in probes1])
        E2, Hvar, Hoth, J2 = st2.Ez[:, mid], st2.Hx[:, mid], st2.Hy[:, mid], st2.Jz[:, mid]
    assert np.max(np.abs(rec1)) > 0.1
    assert np.array_equal(rec2, rec1[0])
    assert np.array_equal(E2, st1.E[0]) and np.array_equal(Hvar, st1.H[0]) and np.array_equal(J2, st1.J[0])
    assert not np.any(Hoth)


# ----------------------------------------------------------------------------- Q2
def _energy2d(E, Hx1, Hx0, Hy1, Hy0, J, wp):
    w = EPS0 * np.sum(E ** 2) + MU0 * (np.sum(Hx1 * Hx0) + np.sum(Hy1 * Hy0))
    pl = wp > 0
    return w + np.sum(J[pl] ** 2 / (EPS0 * wp[pl] ** 2))


@pytest.mark.parametrize("case", ["vacuum", "lossless_plasma", "lossy_plasma"])
def test_Q2_discrete_energy_in_a_conducting_box(case):
    """W^n = eps0 sum Ez^2 + mu0 sum (Hx^{n+1/2} Hx^{n-1/2} + Hy^{n+1/2} Hy^{n-1/2}) + sum Jz^2/(eps0 wp^2) is conserved
    by eqs. (11), (12), (14) when nu = 0 (trapezoidal current, centred curls) and decreases when nu > 0.  A wrong sign or
    index in either curl, or a coefficient of the wrong axis (dx != dy here), breaks it."""
    nx, ny, nsteps = 72, 56, 1500
    dx, dy = DX, 1.4 * DX
    wp = np.zeros((ny, nx)); nu = np.zeros((ny, nx))
    if case != "vacuum":
        wp[20:40, 30:55] = 2 * math.pi * 28.7e9
        wp[5:12, 8:20] = 2 * math.pi * 50e9
    if case == "lossy_plasma":
        nu[wp > 0] = 2e10
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    E0 = np.exp(-((i - 18.0) / 5.0) ** 2 - ((j - 30.0) / 7.0) ** 2)
    E0[0, :] = E0[-1, :] = 0.0; E0[:, 0] = E0[:, -1] = 0.0
    st = oracle.State2D(nx, ny, Ez0=E0)
    W = []
    Hx0, Hy0 = st.Hx.copy(), st.Hy.copy()
    for n in range(nsteps):
        E_n, J_n = st.Ez.copy(), st.Jz.copy()
        oracle.run2d(st, wp, nu, dx, dy, DT, 1, boundary=oracle.BOUNDARY_PEC)
        W.append(_energy2d(E_n, st.Hx, Hx0, st.Hy, Hy0, J_n, wp))
        Hx0, Hy0 = st.Hx.copy(), st.Hy.copy()
    W = np.array(W)
    if case == "lossy_plasma":
        assert np.all(np.diff(W) <= 1e-13 * W[0]) and W[-1] < 0.95 * W[0]
    else:
        assert np.max(np.abs(W / W[0] - 1.0)) < 2e-13


# ----------------------------------------------------------------------------- Q3
def test_Q3_cavity_mode_follows_the_yee_dispersion_relation():
    """Vacuum, conducting box, Ez^0 = sin(m pi i/(nx-1)) sin(n pi j/(ny-1)), H^{-1/2} = 0.  The mode is an eigenvector of
    the discrete curl-curl, so Ez^n = a_n Ez^0 with a_0 = 1, a_1 = 1 - L (H starts from rest half a step early),
    a_{n+1} = (2 - L) a_n - a_{n-1}, L = 4 [(c dt/dx)^2 sin^2(kx dx/2) + (c dt/dy)^2 sin^2(ky dy/2)]
    (Taflove & Hagness, numerical dispersion of the Yee scheme).  The scalar recurrence below shares nothing with the
    grid code; dx != dy and m != n make every exchanged constant visible."""
    nx, ny, m, n, nsteps = 41, 31, 2, 3, 400
    dx, dy = DX, 1.3 * DX
    dt = 0.9 * DT
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    mode = np.sin(m * math.pi * i / (nx - 1)) * np.sin(n * math.pi * j / (ny - 1))
    mode[0, :] = mode[-1, :] = 0.0; mode[:, 0] = mode[:, -1] = 0.0
    L = 4.0 * ((C0 * dt / dx) ** 2 * math.sin(m * math.pi / (2 * (nx - 1))) ** 2 +
               (C0 * dt / dy) ** 2 * math.sin(n * math.pi / (2 * (ny - 1))) ** 2)
    a = [1.0, 1.0 - L]
    for _ in range(nsteps - 1):
        a.append((2.0 - L) * a[-1] - a[-2])
    a = np.array(a)
    st = oracle.State2D(nx, ny, Ez0=mode)
    z = np.zeros((ny, nx))
    probes = [(7, 5), (20, 15), (33, 22), (12, 26)]
    rec, _ = oracle.run2d(st, z, z, dx, dy, dt, nsteps, probes=probes, boundary=oracle.BOUNDARY_PEC)
    assert abs(a).max() <= 1.01 and a.min() < -0.9                   # it really oscillates, several periods
    for p, (pi, pj) in enumerate(probes):
        assert np.max(np.abs(rec[p] - a[1:] * mode[pj, pi])) < 5e-12
    assert np.max(np.abs(st.Ez - a[-1] * mode)) < 5e-12


# ----------------------------------------------------------------------------- Q4
@pytest.mark.parametrize("nu", [0.0, 2e10, 1e11])
def test_Q4_J_is_exact_solution_of_eq6_for_piecewise_linear_E(nu):
    """Same brute force as the 1-D pin P4, through the 2-D code path: RK4 of dJ/dt + nu J = eps0 wp^2 E(t)."""
    nx, ny, nsteps = 60, 50, 300
    wpv = 2 * math.pi * 28.7e9
    wp = np.zeros((ny, nx)); nuv = np.zeros((ny, nx))
    wp[15:40, 30:50] = wpv; nuv[15:40, 30:50] = nu
    st = oracle.State2D(nx, ny)
    rec, recJ = oracle.run2d(st, wp, nuv, DX, DX, DT, nsteps, src_kind=0, src_params=SRC, src_ij=(20, 25),
                             probes=[(35, 27)], record_J=True)
    Es = np.concatenate([[0.0], rec[0]]); Js = np.concatenate([[0.0], recJ[0]])
    assert np.max(np.abs(Js)) > 0
    nsub = 48; h = DT / nsub; J = 0.0; Jref = [0.0]
    for s in range(nsteps):
        e0, e1 = Es[s], Es[s + 1]
        f = lambda t, jv: -nu * jv + EPS0 * wpv ** 2 * (e0 + (e1 - e0) * t / DT)
        for q in range(nsub):
            t = q * h
            k1 = f(t, J); k2 = f(t + h / 2, J + h / 2 * k1); k3 = f(t + h / 2, J + h / 2 * k2); k4 = f(t + h, J + h * k3)
            J += h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        Jref.append(J)
    Jref = np.array(Jref)
    assert np.max(np.abs(Js - Jref)) < 5e-13 * np.max(np.abs(Jref))


# ----------------------------------------------------------------------------- Q5
@pytest.mark.parametrize("boundary", [oracle.BOUNDARY_MUR, oracle.BOUNDARY_PEC])
def test_Q5_exchanging_the_axes_transposes_the_result(boundary):
    nx, ny, nsteps = 64, 45, 260
    dx, dy = DX, 1.25 * DX
    rng = np.random.default_rng(11)
    wp = np.zeros((ny, nx)); nu = np.zeros((ny, nx))
    wp[10:30, 35:60] = 2 * math.pi * 40e9; nu[10:30, 35:60] = 3e10
    E0 = 1e-3 * rng.uniform(-1, 1, (ny, nx))
    probes = [(20, 22), (40, 15), (1, 30), (50, 1), (0, 7), (63, 20), (30, 44), (33, 0)]
    a = oracle.State2D(nx, ny, Ez0=E0)
    ra, _ = oracle.run2d(a, wp, nu, dx, dy, DT, nsteps, src_kind=0, src_params=SRC, src_ij=(20, 22), probes=probes,
                         boundary=boundary)
    b = oracle.State2D(ny, nx, Ez0=E0.T)
    rb, _ = oracle.run2d(b, wp.T.copy(), nu.T.copy(), dy, dx, DT, nsteps, src_kind=0, src_params=SRC, src_ij=(22, 20),
                         probes=[(j, i) for i, j in probes], boundary=boundary)
    scale = np.max(np.abs(ra))
    assert scale > 5e-3
    assert np.max(np.abs(ra - rb)) < 1e-13 * scale
    assert np.max(np.abs(a.Ez - b.Ez.T)) < 1e-13 * scale
    # H is a pseudo-vector: exchanging x and y maps Hx -> -Hy, Hy -> -Hx
    hs = np.max(np.abs(a.Hx))
    assert np.max(np.abs(a.Hx + b.Hy.T)) < 1e-13 * hs and np.max(np.abs(a.Hy + b.Hx.T)) < 1e-13 * hs


def test_Q5b_point_source_in_a_uniform_medium_keeps_the_square_symmetries():
    n, nsteps = 61, 100
    c = n // 2
    wp = np.full((n, n), 2 * math.pi * 20e9); nu = np.full((n, n), 1e10)
    st = oracle.State2D(n, n)
    oracle.run2d(st, wp, nu, DX, DX, DT, nsteps, src_kind=0, src_params=SRC, src_ij=(c, c))
    E = st.Ez
    s = np.max(np.abs(E))
    assert s > 1e-3
    for other in (E[::-1, :], E[:, ::-1], E.T):
        assert np.max(np.abs(E - other)) < 1e-12 * s


# ----------------------------------------------------------------------------- Q6: Mur, soft source, timing
def test_Q6_source_probe_timing_and_first_steps_by_hand():
    """Vacuum, one unit sample added at step 0 at (is, js): sample 0 of a probe there reads 1, and one step later the
    four neighbours read (c dt/dx)^2 resp. (c dt/dy)^2 and the node itself 1 - 2 (Sx^2 + Sy^2) (five-point Laplacian)."""
    nx, ny = 21, 17
    dx, dy = DX, 2.0 * DX
    sx2, sy2 = (C0 * DT / dx) ** 2, (C0 * DT / dy) ** 2
    z = np.zeros((ny, nx))
    st = oracle.State2D(nx, ny)
    rec, _ = oracle.run2d(st, z, z, dx, dy, DT, 2, src_kind=oracle.SRC_TABLE, src_params=(1.0,), src_ij=(9, 8),
                          probes=[(9, 8), (10, 8), (8, 8), (9, 9), (9, 7), (10, 9)])
    assert rec[0, 0] == 1.0 and not np.any(rec[1:, 0])
    assert rec[0, 1] == pytest.approx(1.0 - 2 * (sx2 + sy2), rel=1e-14)
    assert rec[1, 1] == pytest.approx(sx2, rel=1e-14) and rec[2, 1] == pytest.approx(sx2, rel=1e-14)
    assert rec[3, 1] == pytest.approx(sy2, rel=1e-14) and rec[4, 1] == pytest.approx(sy2, rel=1e-14)
    assert rec[5, 1] == 0.0


def test_Q6b_mur_edges_absorb_and_beat_the_conductor():
    """Echo = record at the source node minus the record of a grid so large that nothing returns in time.  The paper's
    pulse (tau = 15 dt); first-order Mur leaves 0.5 % of the pulse peak, the conductor 19 %."""
    nsteps = 600
    src = (15 * DT, 75 * DT, 1.0)

    def record(nx, ny, bc):
        z = np.zeros((ny, nx))
        st = oracle.State2D(nx, ny)
        rec, _ = oracle.run2d(st, z, z, DX, DX, DT, nsteps, src_kind=0, src_params=src, src_ij=(nx // 2, ny // 2),
                              probes=[(nx // 2, ny // 2)], boundary=bc)
        return rec[0]

    ref = record(340, 340, oracle.BOUNDARY_PEC)            # edges 170 nodes away: an echo needs 680 steps
    echo_mur = np.max(np.abs(record(200, 160, oracle.BOUNDARY_MUR) - ref))
    echo_pec = np.max(np.abs(record(200, 160, oracle.BOUNDARY_PEC) - ref))
    assert echo_pec > 0.1 * np.max(np.abs(ref))
    assert echo_mur < 0.05 * echo_pec


# ----------------------------------------------------------------------------- Q7
def test_Q7_domain_of_dependence_window_is_bit_exact():
    w = wl.tm2d_column(nx=220, ny=180, nsteps=40)
    full = oracle.run_workload2d(w)
    pi, pj = (int(v) for v in w.probes[4])                 # the grid centre
    m = w.nsteps + 1
    win = oracle.run_workload2d(w, window=(pi - m, pi + m + 1, pj - m, pj + m + 1))
    k = [tuple(p) for p in full["probe_ij"]].index((pi, pj))
    kw = [tuple(p) for p in win["probe_ij"]].index((pi, pj))
    assert np.max(np.abs(full["rec"][k])) > 0
    assert np.array_equal(full["rec"][k], win["rec"][kw])


# ----------------------------------------------------------------------------- Q8
def test_Q8_openmp_build_is_bit_identical():
    w = wl.tm2d_column(nx=150, ny=90, nsteps=120)
    a = oracle.run_workload2d(w, omp=False)
    b = oracle.run_workload2d(w, omp=True)
    assert np.array_equal(a["rec"], b["rec"]) and np.array_equal(a["state"].Ez, b["state"].Ez)
    assert np.array_equal(a["state"].Jz, b["state"].Jz) and np.array_equal(a["state"].Hx, b["state"].Hx)


def test_Q9_run_is_restartable_and_arguments_are_checked():
    w = wl.tm2d_column(nx=40, ny=30, nsteps=30)
    a = oracle.run_workload2d(w)
    wp, nu = w.media()
    st = oracle.State2D(w.nx, w.ny, Ez0=w.initial_E())
    kw = dict(src_kind=w.src_kind, src_params=w.src_params, src_ij=w.src_ij, probes=w.probes)
    r1, _ = oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, 13, **kw)
    r2, _ = oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, 17, **kw)
    assert np.array_equal(np.concatenate([r1, r2], 1), a["rec"])
    with pytest.raises(ValueError):
        oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, 1, probes=[(w.nx, 0)])
    with pytest.raises(ValueError):
        oracle.run2d(st, wp, nu, w.dx, w.dy, w.dt, 1, src_kind=0, src_params=SRC, src_ij=(0, w.ny))


# ============================================================================ the paper's boundary in 2-D: split-field PML
PML2 = (8, 2.0, 1e-4)


@pytest.mark.parametrize("axis", ["x", "y"])
def test_U1_pml_uniform_along_one_axis_is_the_1d_pml_oracle_bit_for_bit(axis):
    """Fields uniform along one axis excite only the split part of the other axis: what is left is the 1-D method with
    the 1-D layer at both ends — same tables, same node depths (E nodes at (npml-k)/npml, H nodes half
    a node deeper), same conductor behind.  Pins every index of the per-axis tables and which part carries which curl."""
    n, nother, nsteps = 300, 2 * 120 + 9, 110
    dvar, doth = DX, 1.7 * DX
    wp1, nu1 = _slab_media_1d(n, 140, 190)
    k = np.arange(n, dtype=np.float64)
    E1 = np.exp(-((k - 60.0) / 9.0) ** 2) * ((k >= PML2[0]) & (k <= n - 1 - PML2[0]))     # nothing inside the layers at t = 0
    st1 = oracle.State(n, 1, E0=E1)
    probes1 = [0, 1, 3, 7, 8, 60, 150, n - 9, n - 2, n - 1]
    rec1, _ = oracle.run(st1, wp1[None], nu1[None], dvar, DT, nsteps, probes=probes1, boundary=oracle.BOUNDARY_PML, pml=PML2)
    mid = nother // 2
    if axis == "x":
        rep = lambda a: np.repeat(a[None, :], nother, 0)
        st2 = oracle.State2D(n, nother, Ez0=rep(E1))
        rec2 = oracle.run2d_pml(st2, rep(wp1), rep(nu1), dvar, doth, DT, nsteps, pml=PML2, probes=[(p, mid) for p in probes1])
        E2, Hvar, J2 = st2.Ez[mid], -st2.Hy[mid], st2.Jz[mid]
    else:
        rep = lambda a: np.repeat(a[:, None], nother, 1)
        st2 = oracle.State2D(nother, n, Ez0=rep(E1))
        rec2 = oracle.run2d_pml(st2, rep(wp1), rep(nu1), doth, dvar, DT, nsteps, pml=PML2, probes=[(mid, p) for p in probes1])
        E2, Hvar, J2 = st2.Ez[:, mid], st2.Hx[:, mid], st2.Jz[:, mid]
    assert np.max(np.abs(rec1)) > 0.1 and np.max(np.abs(rec1[0][3])) > 1e-3          # the pulse has entered the left layer
    assert np.array_equal(rec2, rec1[0])
    assert np.array_equal(E2, st1.E[0]) and np.array_equal(Hvar, st1.H[0]) and np.array_equal(J2, st1.J[0])


def test_U2_pml_with_R0_one_is_the_conducting_box():
    """R0 = 1: sigma = 0 everywhere, the split parts add up to the unsplit vacuum update (up to the rounding of the sum
    Ezx + Ezy) and the four edges are the conductor: the run equals oracle2d_run with BOUNDARY_PEC when the nodes that
    would be layer are vacuum."""
    nx, ny, nsteps = 70, 56, 200
    wp = np.zeros((ny, nx)); nu = np.zeros((ny, nx))
    wp[25:35, 30:45] = 2 * math.pi * 28.7e9; nu[25:35, 30:45] = 2e10
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    E0 = np.exp(-((i - 20.0) / 4.0) ** 2 - ((j - 30.0) / 5.0) ** 2)
    E0[0, :] = E0[-1, :] = 0.0; E0[:, 0] = E0[:, -1] = 0.0
    a = oracle.State2D(nx, ny, Ez0=E0)
    ra = oracle.run2d_pml(a, wp, nu, DX, 1.3 * DX, 0.9 * DT, nsteps, pml=(6, 2.0, 1.0), probes=[(35, 28), (3, 3), (60, 50)])
    b = oracle.State2D(nx, ny, Ez0=E0)
    rb, _ = oracle.run2d(b, wp, nu, DX, 1.3 * DX, 0.9 * DT, nsteps, probes=[(35, 28), (3, 3), (60, 50)], boundary=oracle.BOUNDARY_PEC)
    assert np.max(np.abs(rb)) > 0.05
    assert np.max(np.abs(ra - rb)) <= 1e-13 * np.max(np.abs(rb))
    assert np.max(np.abs(a.Ez - b.Ez)) <= 1e-13 * np.max(np.abs(b.Ez)) and np.max(np.abs(a.Jz - b.Jz)) <= 1e-13 * np.max(np.abs(b.Jz))


def test_U3_pml_absorbs_an_oblique_pulse_better_than_first_order_mur_and_never_feeds_energy():
    """A point-like pulse next to a corner: its circular wavefront meets the sides at every angle.  Peak of what comes back
    to a probe in the middle, relative to the direct pulse: the layer (10 nodes) beats first-order Mur, which is exact at
    normal incidence only; and the field energy of the lossless vacuum run only goes down once the front is in the layer."""
    nx, ny, nsteps = 161, 161, 700
    z = np.zeros((ny, nx))
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    E0 = np.exp(-((i - 40.0) / 3.0) ** 2 - ((j - 40.0) / 3.0) ** 2)
    probe = [(80, 80)]
    a = oracle.State2D(nx, ny, Ez0=E0)
    ra = oracle.run2d_pml(a, z, z, DX, DX, DT, nsteps, pml=(10, 3.0, 1e-6), probes=probe)[0]
    b = oracle.State2D(nx, ny, Ez0=E0)
    rb = oracle.run2d(b, z, z, DX, DX, DT, nsteps, probes=probe, boundary=oracle.BOUNDARY_MUR)[0][0]
    big = oracle.State2D(3 * nx, 3 * ny, Ez0=np.pad(E0, ((ny, ny), (nx, nx))))           # no boundary within reach: the reference
    rr = oracle.run2d(big, np.zeros((3 * ny, 3 * nx)), np.zeros((3 * ny, 3 * nx)), DX, DX, DT, nsteps,
                      probes=[(80 + nx, 80 + ny)], boundary=oracle.BOUNDARY_PEC)[0][0]
    direct = np.max(np.abs(rr))
    err_pml, err_mur = np.max(np.abs(ra - rr)) / direct, np.max(np.abs(rb - rr)) / direct
    print(f"reflection seen at the probe: PML(10) {err_pml:.2e}, Mur-1 {err_mur:.2e}")
    assert direct > 1e-2 and err_pml < 0.25 * err_mur and err_pml < 5e-3
    c = oracle.State2D(nx, ny, Ez0=E0)
    W = []
    Hx0, Hy0 = c.Hx.copy(), c.Hy.copy()
    for n in range(300):
        E_n = c.Ez.copy()
        oracle.run2d_pml(c, z, z, DX, DX, DT, 1, pml=(10, 3.0, 1e-6))
        W.append(EPS0 * np.sum(E_n ** 2) + MU0 * (np.sum(c.Hx * Hx0) + np.sum(c.Hy * Hy0)))
        Hx0, Hy0 = c.Hx.copy(), c.Hy.copy()
    W = np.array(W)
    assert np.all(np.diff(W) <= 1e-12 * W[0]) and W[-1] < 0.5 * W[0]


def test_U4_pml_restart_and_argument_checks():
    nx, ny = 60, 50
    rng = np.random.default_rng(6)
    wp = rng.uniform(0, 2 * math.pi * 40e9, (ny, nx)); nu = rng.uniform(0, 5e10, (ny, nx))
    E0 = rng.uniform(-1, 1, (ny, nx))
    a = oracle.State2D(nx, ny, Ez0=E0)
    ra = oracle.run2d_pml(a, wp, nu, DX, DX, DT, 60, pml=PML2, src_kind=0, src_params=SRC, src_ij=(3, 20), probes=[(3, 20), (30, 25)])
    out = []
    for omp in (False, True):
        b = oracle.State2D(nx, ny, Ez0=E0)
        r1 = oracle.run2d_pml(b, wp, nu, DX, DX, DT, 25, pml=PML2, src_kind=0, src_params=SRC, src_ij=(3, 20), probes=[(3, 20), (30, 25)], omp=omp)
        r2 = oracle.run2d_pml(b, wp, nu, DX, DX, DT, 35, pml=PML2, src_kind=0, src_params=SRC, src_ij=(3, 20), probes=[(3, 20), (30, 25)], omp=omp)
        out.append(np.concatenate([r1, r2], 1))
        assert np.array_equal(a.Ez, b.Ez) and np.array_equal(a.Esplit, b.Esplit) and np.array_equal(a.Jz, b.Jz)
    assert np.array_equal(out[0], ra) and np.array_equal(out[1], ra)
    assert not np.any(a.Jz[:PML2[0]]) and not np.any(a.Jz[:, -PML2[0]:])              # layer nodes carry no current
    c = oracle.State2D(nx, ny)
    for bad in ((0, 2.0, 1e-4), (30, 2.0, 1e-4), (5, 2.0, 0.0), (5, -1.0, 1e-4)):
        with pytest.raises(ValueError):
            oracle.run2d_pml(c, wp, nu, DX, DX, DT, 1, pml=bad)
