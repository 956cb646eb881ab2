"""Pins for the 2-D TEz half of the CPU oracle (oracle/rketd_oracle.cpp, oracle2d_te_run) — SURVEY §8(f) NEXT-3
("2-D TMz/TEz").  The paper gives the vector equations (1)-(3) and prints nothing 2-D; what fixes
the TEz oracle is: its reduction to the (pinned) 1-D oracle when the fields do not vary along one axis (R1, both
axes: Ey, Hz along x; Ex, -Hz along y), the energy invariant of the lossless leapfrog in a conducting box (R2), the
TE_mn eigenmodes of that box, which follow the Yee dispersion relation exactly (R3, dx != dy, m != n), the symmetry
under exchange of the axes (R4), the first step worked out by hand (R5), the domain of dependence (R6) and
OpenMP == serial (R7).  None of these tests touches the CUDA path.
"""
import math

import numpy as np
import pytest

import oracle

C0, MU0, EPS0 = oracle.constants()
DX = 75e-6
DT = DX / (2 * C0)


def _slab_media_1d(n, lo, hi, wp0=2 * math.pi * 28.7e9, nu0=2e10):
    wp = np.zeros(n); nu = np.zeros(n)
    wp[lo:hi] = wp0; nu[lo:hi] = nu0
    return wp, nu


# ----------------------------------------------------------------------------- R1
@pytest.mark.parametrize("axis", ["x", "y"])
def test_R1_uniform_along_one_axis_is_the_1d_oracle_bit_for_bit(axis):
    """Along x: (Ey, Hz, Jy) are (E, H, J) of the 1-D method, Ex stays 0.  Along y: (Ex, -Hz, Jx) are (E, H, J), Ey
    stays 0.  Away from the edges of the uniform axis (a disturbance travels one node per step) the match is exact:
    every index, sign, coefficient-of-which-axis and the order of S1-S6 is pinned to the pinned 1-D oracle."""
    n, nother, nsteps = 300, 2 * 120 + 9, 110
    dvar, doth = DX, 1.7 * DX
    wp1, nu1 = _slab_media_1d(n, 140, 190)
    k = np.arange(n, dtype=np.float64)
    E1 = np.exp(-((k - 100.0) / 12.0) ** 2)
    rng = np.random.default_rng(5)
    H1 = 1e-3 * rng.uniform(-1, 1, n); H1[-1] = 0.0
    J1 = 1e-2 * rng.uniform(-1, 1, n) * (wp1 > 0)
    tab = rng.uniform(-1, 1, 60)
    st1 = oracle.State(n, 1, E0=E1, H0=H1, J0=J1)
    probes1 = [0, 1, 60, 150, 189, n - 2, n - 1]
    rec1, _ = oracle.run(st1, wp1[None], nu1[None], dvar, DT, nsteps, probes=probes1, src_kind=oracle.SRC_TABLE,
                         src_params=tab, src_cell=77)
    mid = nother // 2
    if axis == "x":    # arrays [ny = nother][nx = n]; the source is a line source: every row is driven alike
        rep = lambda a: np.repeat(a[None, :], nother, 0)
        st2 = oracle.State2DTE(n, nother, Ey0=rep(E1), Hz0=rep(H1), Jy0=rep(J1))
        recs = []
        for s in range(nsteps):      # a line source = the point source of every row: step by step, adding it by hand
            oracle.run2d_te(st2, rep(wp1), rep(nu1), dvar, doth, DT, 1)
            if s < len(tab):
                st2.Ey[:, 77] += tab[s]
                # J' was formed from E' before the source was added: redo eq. (11)'s last term for the driven column
                cf = oracle.coefficients(wp1[77:78], nu1[77:78], dvar, DT)
                st2.Jy[:, 77] += cf["kc"][0] * tab[s]
            recs.append([st2.Ey[mid, p] for p in probes1])
        rec2 = np.array(recs).T
        E2, Hvar, Eoth, J2 = st2.Ey[mid], st2.Hz[mid], st2.Ex[mid], st2.Jy[mid]
        assert wp1[77] == 0.0          # the driven column is vacuum: kc = 0, the J correction above is exactly 0
    else:              # arrays [ny = n][nx = nother]
        rep = lambda a: np.repeat(a[:, None], nother, 1)
        st2 = oracle.State2DTE(nother, n, Ex0=rep(E1), Hz0=rep(-H1), Jx0=rep(J1))
        recs = []
        for s in range(nsteps):
            oracle.run2d_te(st2, rep(wp1), rep(nu1), doth, dvar, DT, 1)
            if s < len(tab):
                st2.Ex[77, :] += tab[s]
            recs.append([st2.Ex[p, mid] for p in probes1])
        rec2 = np.array(recs).T
        E2, Hvar, Eoth, J2 = st2.Ex[:, mid], -st2.Hz[:, mid], st2.Ey[:, mid], st2.Jx[:, mid]
    assert np.max(np.abs(rec1)) > 0.1
    assert np.array_equal(rec2, rec1[0])
    assert np.array_equal(E2, st1.E[0]) and np.array_equal(Hvar, st1.H[0]) and np.array_equal(J2, st1.J[0])
    assert not np.any(Eoth)


def test_R1b_point_source_and_probe_components():
    """The soft source drives the component asked for at the node asked for, sample s((n+1) dt) at step n, and a probe
    reads the component asked for (first steps, vacuum)."""
    nx, ny = 21, 17
    z = np.zeros((ny, nx))
    for comp in (oracle.EX, oracle.EY):
        st = oracle.State2DTE(nx, ny)
        tab = [0.5, -0.25, 0.125]
        rec = oracle.run2d_te(st, z, z, DX, 1.3 * DX, DT, 1, src_kind=oracle.SRC_TABLE, src_params=tab, src_ij=(9, 8),
                              src_comp=comp, probes=[(9, 8, oracle.EX), (9, 8, oracle.EY), (10, 8, comp)])
        assert rec[comp, 0] == 0.5 and rec[1 - comp, 0] == 0.0 and rec[2, 0] == 0.0
        assert (st.Ex if comp == oracle.EX else st.Ey)[8, 9] == 0.5 and not np.any(st.Hz)


# ----------------------------------------------------------------------------- R2
def _energy_te(Ex, Ey, Hz1, Hz0, Jx, Jy, wp):
    w = EPS0 * (np.sum(Ex ** 2) + np.sum(Ey ** 2)) + MU0 * np.sum(Hz1 * Hz0)
    pl = wp > 0
    return w + np.sum((Jx[pl] ** 2 + Jy[pl] ** 2) / (EPS0 * wp[pl] ** 2))


@pytest.mark.parametrize("case", ["vacuum", "lossless_plasma", "lossy_plasma"])
def test_R2_discrete_energy_in_a_conducting_box(case):
    """W^n = eps0 sum (Ex^2 + Ey^2) + mu0 sum Hz^{n+1/2} Hz^{n-1/2} + sum (Jx^2 + Jy^2)/(eps0 wp^2) is conserved when nu = 0
    and decreases when nu > 0.  A wrong sign or index in either curl term, or the coefficient of the wrong axis
    (dx != dy), breaks it."""
    nx, ny, nsteps = 72, 56, 700
    dx, dy = DX, 1.4 * DX
    wp = np.zeros((ny, nx)); nu = np.zeros((ny, nx))
    if case != "vacuum":
        wp[20:40, 30:55] = 2 * math.pi * 28.7e9
        wp[5:12, 8:20] = 2 * math.pi * 50e9
    if case == "lossy_plasma":
        nu[wp > 0] = 2e10
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    Hz0 = np.exp(-((i - 18.0) / 5.0) ** 2 - ((j - 30.0) / 7.0) ** 2)
    Hz0[-1, :] = 0.0; Hz0[:, -1] = 0.0                      # padding row / column
    st = oracle.State2DTE(nx, ny, Hz0=Hz0)
    W = []
    Hprev = st.Hz.copy()
    for n in range(nsteps):
        Ex_n, Ey_n, Jx_n, Jy_n = st.Ex.copy(), st.Ey.copy(), st.Jx.copy(), st.Jy.copy()
        oracle.run2d_te(st, wp, nu, dx, dy, DT, 1, boundary=oracle.BOUNDARY_PEC)
        if n > 0:
            W.append(_energy_te(Ex_n, Ey_n, st.Hz, Hprev, Jx_n, Jy_n, wp))
        Hprev = st.Hz.copy()
    W = np.array(W)
    assert W[0] > 0
    if case == "lossy_plasma":
        assert np.all(np.diff(W) <= 1e-13 * W[0]) and W[-1] < 0.97 * W[0]
    else:
        assert np.max(np.abs(W / W[0] - 1.0)) < 2e-13


# ----------------------------------------------------------------------------- R3
def test_R3_cavity_mode_follows_the_yee_dispersion_relation():
    """Vacuum, conducting box.  Hz^{-1/2} = cos(m pi (i+1/2)/(nx-1)) cos(n pi (j+1/2)/(ny-1)), E^0 = 0: the TE_mn mode is an
    eigenvector of the discrete curl-curl, so Hz^{k-1/2} = a_k Hz^{-1/2} with a_0 = a_1 = 1 (E starts from rest),
    a_{k+1} = (2 - L) a_k - a_{k-1}, L = 4 [(c dt/dx)^2 sin^2(kx dx/2) + (c dt/dy)^2 sin^2(ky dy/2)] (numerical dispersion
    of the Yee scheme).  The scalar recurrence shares nothing with the grid code."""
    nx, ny, m, n, nsteps = 41, 31, 2, 3, 400
    dx, dy = DX, 1.3 * DX
    dt = 0.9 * DT
    i = np.arange(nx)[None, :]; j = np.arange(ny)[:, None]
    mode = np.cos(m * math.pi * (i + 0.5) / (nx - 1)) * np.cos(n * math.pi * (j + 0.5) / (ny - 1))
    mode[-1, :] = 0.0; mode[:, -1] = 0.0
    L = 4.0 * ((C0 * dt / dx) ** 2 * math.sin(m * math.pi / (2 * (nx - 1))) ** 2 +
               (C0 * dt / dy) ** 2 * math.sin(n * math.pi / (2 * (ny - 1))) ** 2)
    a = [1.0, 1.0]
    for _ in range(nsteps):
        a.append((2.0 - L) * a[-1] - a[-2])
    st = oracle.State2DTE(nx, ny, Hz0=mode)
    z = np.zeros((ny, nx))
    worst = 0.0
    for k in range(1, nsteps + 1):
        oracle.run2d_te(st, z, z, dx, dy, dt, 1, boundary=oracle.BOUNDARY_PEC)
        worst = max(worst, np.max(np.abs(st.Hz - a[k] * mode)))
    assert min(a) < -0.9 and worst < 5e-12


# ----------------------------------------------------------------------------- R4
def test_R4_exchanging_the_axes_transposes_the_result():
    """(x, y) -> (y, x) maps (Ex, Ey, Hz) -> (Ey^T, Ex^T, -Hz^T): the transposed problem gives the transposed fields, up to
    rounding (S1 adds its two curl terms in a fixed order, so the images differ in the last bits; an exchanged constant
    or a wrong sign shows at the 1e-1 level with dx = 1.6 dy)."""
    nx, ny, nsteps = 50, 37, 90
    dx, dy = DX, 1.6 * DX
    rng = np.random.default_rng(8)
    wp = rng.uniform(0, 2 * math.pi * 40e9, (ny, nx)) * (rng.uniform(size=(ny, nx)) > 0.5)
    nu = rng.uniform(0, 5e10, (ny, nx))
    Ex0 = rng.uniform(-1, 1, (ny, nx)); Ex0[:, -1] = 0.0
    Ey0 = rng.uniform(-1, 1, (ny, nx)); Ey0[-1, :] = 0.0
    Hz0 = 1e-3 * rng.uniform(-1, 1, (ny, nx)); Hz0[-1, :] = 0.0; Hz0[:, -1] = 0.0
    sa = oracle.State2DTE(nx, ny, Ex0=Ex0, Ey0=Ey0, Hz0=Hz0)
    ra = oracle.run2d_te(sa, wp, nu, dx, dy, DT, nsteps, src_kind=0, src_params=(2e-12, 6e-12, 1.0), src_ij=(20, 11),
                         src_comp=oracle.EX, probes=[(7, 30, oracle.EX), (44, 3, oracle.EY)])
    sb = oracle.State2DTE(ny, nx, Ex0=Ey0.T, Ey0=Ex0.T, Hz0=-Hz0.T)
    rb = oracle.run2d_te(sb, wp.T, nu.T, dy, dx, DT, nsteps, src_kind=0, src_params=(2e-12, 6e-12, 1.0), src_ij=(11, 20),
                         src_comp=oracle.EY, probes=[(30, 7, oracle.EY), (3, 44, oracle.EX)])
    close = lambda a, b: np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(a))
    assert np.max(np.abs(ra)) > 0.1 and close(ra, rb)
    assert close(sa.Ex, sb.Ey.T) and close(sa.Ey, sb.Ex.T) and close(sa.Hz, -sb.Hz.T)
    assert close(sa.Jx, sb.Jy.T) and close(sa.Jy, sb.Jx.T)


# ----------------------------------------------------------------------------- R5
def test_R5_first_steps_by_hand_and_mur_echo():
    """One Hz impulse in vacuum.  Step 1: Hz unchanged (E = 0); Ex' = +cey (Hz[j] - Hz[j-1]) -> +cey at (i, j), -cey at
    (i, j+1); Ey' = -cex (Hz[i] - Hz[i-1]) -> -cex at (i, j), +cex at (i+1, j).  Step 2: the centre loses
    2 chx cex + 2 chy cey (the five-point Laplacian of the scalar wave equation Hz obeys)."""
    nx, ny = 15, 13
    dx, dy = DX, 1.25 * DX
    z = np.zeros((ny, nx))
    Hz0 = z.copy(); Hz0[6, 7] = 1.0
    st = oracle.State2DTE(nx, ny, Hz0=Hz0)
    cf = oracle.coefficients2d(z[0], z[0], dx, dy, DT)
    cex, cey, chx, chy = cf["cex"][0], cf["cey"][0], cf["chx"], cf["chy"]
    oracle.run2d_te(st, z, z, dx, dy, DT, 1)
    assert np.array_equal(st.Hz, Hz0)
    Ex_expect = z.copy(); Ex_expect[6, 7] = cey; Ex_expect[7, 7] = -cey
    Ey_expect = z.copy(); Ey_expect[6, 7] = -cex; Ey_expect[6, 8] = cex
    assert np.array_equal(st.Ex, Ex_expect) and np.array_equal(st.Ey, Ey_expect)
    oracle.run2d_te(st, z, z, dx, dy, DT, 1)
    assert abs(st.Hz[6, 7] - (1.0 - 2 * chx * cex - 2 * chy * cey)) < 1e-15
    assert abs(st.Hz[6, 8] - chx * cex) < 1e-16 and abs(st.Hz[7, 7] - chy * cey) < 1e-16
    assert abs(st.Hz[6, 6] - chx * cex) < 1e-16 and abs(st.Hz[5, 7] - chy * cey) < 1e-16
    # Mur absorbs a plane pulse that a conductor reflects whole
    n = 400
    k = np.arange(n, dtype=np.float64)
    Ey0 = np.repeat(np.exp(-((k - 300.0) / 15.0) ** 2)[None, :], 9, 0)
    Hz0 = np.repeat((np.exp(-((k + 0.5 - 300.0) / 15.0) ** 2) / (MU0 * C0))[None, :], 9, 0)
    Hz0[:, -1] = 0.0; Hz0[-1, :] = 0.0
    zz = np.zeros((9, n))
    echo = {}
    for bc in (oracle.BOUNDARY_MUR, oracle.BOUNDARY_PEC):
        st = oracle.State2DTE(n, 9, Ey0=Ey0, Hz0=Hz0)
        rec = oracle.run2d_te(st, zz, zz, DX, DX, DT, 600, probes=[(200, 4, oracle.EY)], boundary=bc)
        echo[bc] = np.max(np.abs(rec[0, 350:]))           # after the pulse has passed node 200 going right... and come back
    assert echo[oracle.BOUNDARY_PEC] > 0.3 and echo[oracle.BOUNDARY_MUR] < 0.02 * echo[oracle.BOUNDARY_PEC]


# ----------------------------------------------------------------------------- R6
def test_R6_windowed_run_is_bit_identical_inside_the_domain_of_dependence():
    nx, ny, nsteps = 140, 120, 30
    rng = np.random.default_rng(3)
    wp = rng.uniform(0, 2 * math.pi * 40e9, (ny, nx)); nu = rng.uniform(0, 5e10, (ny, nx))
    Ex0 = rng.uniform(-1, 1, (ny, nx)); Ex0[:, -1] = 0.0
    Ey0 = rng.uniform(-1, 1, (ny, nx)); Ey0[-1, :] = 0.0
    full = oracle.State2DTE(nx, ny, Ex0=Ex0, Ey0=Ey0)
    pi, pj = 70, 60
    rf = oracle.run2d_te(full, wp, nu, DX, DX, DT, nsteps, probes=[(pi, pj, oracle.EX), (pi, pj, oracle.EY)])
    r = nsteps + 2
    i0, i1, j0, j1 = pi - r, pi + r + 1, pj - r, pj + r + 1
    ex = Ex0[j0:j1, i0:i1].copy(); ey = Ey0[j0:j1, i0:i1].copy()
    win = oracle.State2DTE(i1 - i0, j1 - j0, Ex0=ex, Ey0=ey)
    rw = oracle.run2d_te(win, wp[j0:j1, i0:i1], nu[j0:j1, i0:i1], DX, DX, DT, nsteps,
                         probes=[(pi - i0, pj - j0, oracle.EX), (pi - i0, pj - j0, oracle.EY)])
    assert np.max(np.abs(rf)) > 0 and np.array_equal(rf, rw)
    assert full.Ex[pj, pi] == win.Ex[pj - j0, pi - i0] and full.Jy[pj, pi] == win.Jy[pj - j0, pi - i0]


# ----------------------------------------------------------------------------- R7
def test_R7_openmp_build_is_bit_identical_and_arguments_are_checked():
    nx, ny = 64, 48
    rng = np.random.default_rng(2)
    wp = rng.uniform(0, 2 * math.pi * 40e9, (ny, nx)); nu = rng.uniform(0, 5e10, (ny, nx))
    Ey0 = rng.uniform(-1, 1, (ny, nx)); Ey0[-1, :] = 0.0
    out = []
    for omp in (False, True):
        st = oracle.State2DTE(nx, ny, Ey0=Ey0)
        rec = oracle.run2d_te(st, wp, nu, DX, 1.2 * DX, DT, 80, src_kind=0, src_params=(2e-12, 6e-12, 1.0), src_ij=(30, 20),
                              probes=[(10, 10, oracle.EY), (50, 30, oracle.EX)], omp=omp)
        out.append((rec, st.Ex.copy(), st.Ey.copy(), st.Hz.copy(), st.Jx.copy(), st.Jy.copy()))
    assert all(np.array_equal(a, b) for a, b in zip(*out))
    st = oracle.State2DTE(nx, ny)
    with pytest.raises(ValueError):
        oracle.run2d_te(st, wp, nu, DX, DX, DT, 1, probes=[(nx, 0, oracle.EX)])
    with pytest.raises(ValueError):
        oracle.run2d_te(st, wp, nu, DX, DX, DT, 1, src_kind=0, src_params=(1e-12, 1e-12, 1.0), src_ij=(0, 0), src_comp=2)
