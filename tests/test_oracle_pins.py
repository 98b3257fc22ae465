"""Pins for the oracle (oracle/hlb_oracle.cpp): things the mathematics fixes.

The paper (arxiv 1906.11925) prints no flow values, so none of these is a paper number;
each is a closed form, an invariant, a brute-force twin or a special case, chosen so that
a dropped term, a wrong sign/index or a transposed direction fails at least one.
Numbering P1..P12 follows SURVEY.md §8(c) "What pins the oracle".
"""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
import workloads as W

C, WT, OPP = oracle.velocity_set()
NQ = 15


@pytest.fixture(autouse=True, params=["d3q15", "d3q19"])
def lattice(request, monkeypatch):
    """Every pin runs for both lattices of the oracle: D3Q15 (BASELINE.json) and D3Q19 (the
    lattice the paper names). The fixture makes `lattice=...` the
    default of oracle.Oracle / oracle.dense_run and points C, WT, OPP, NQ at that lattice."""
    import sys
    lat = request.param
    orig_init, orig_dense = oracle.Oracle.__init__, oracle.dense_run

    def init(self, *a, **k):
        k.setdefault("lattice", lat)
        orig_init(self, *a, **k)

    def dense(*a, **k):
        k.setdefault("lattice", lat)
        return orig_dense(*a, **k)

    monkeypatch.setattr(oracle.Oracle, "__init__", init)
    monkeypatch.setattr(oracle, "dense_run", dense)
    me = sys.modules[__name__]
    c, w, o = oracle.velocity_set(lat)
    monkeypatch.setattr(me, "C", c)
    monkeypatch.setattr(me, "WT", w)
    monkeypatch.setattr(me, "OPP", o)
    monkeypatch.setattr(me, "NQ", len(w))
    return lat


def canon_coords(st):
    nz, ny, nx = st.shape
    v = np.flatnonzero(st.reshape(-1) == 1)
    return v % nx, (v // nx) % ny, v // (nx * ny)


# ------------------------------------------------------------------ P1 lattice identities
def test_p1_velocity_set_is_d3q15_or_d3q19(lattice):
    vecs = {tuple(int(a) for a in c) for c in C}
    assert len(vecs) == NQ == {"d3q15": 15, "d3q19": 19}[lattice]
    assert (0, 0, 0) in vecs
    axis = {v for v in vecs if sum(abs(a) for a in v) == 1}
    cube = {v for v in vecs if all(abs(a) == 1 for a in v)}
    face = {v for v in vecs if sum(abs(a) for a in v) == 2}
    assert len(axis) == 6
    if lattice == "d3q15":
        assert len(cube) == 8 and len(face) == 0
        table = {0: Fraction(2, 9), 1: Fraction(1, 9), 3: Fraction(1, 72)}
    else:
        assert len(cube) == 0 and len(face) == 12
        table = {0: Fraction(1, 3), 1: Fraction(1, 18), 2: Fraction(1, 36)}
    w = [Fraction(float(x)).limit_denominator(1000) for x in WT]
    for c, wq in zip(C, w):
        assert wq == table[int(np.dot(c, c))]
    assert sum(w) == 1


def test_p1_moment_identities():
    w = [Fraction(float(x)).limit_denominator(1000) for x in WT]
    c = [[int(a) for a in q] for q in C]
    d = lambda a, b: 1 if a == b else 0
    for a in range(3):
        assert sum(w[q] * c[q][a] for q in range(NQ)) == 0
        for b in range(3):
            assert sum(w[q] * c[q][a] * c[q][b] for q in range(NQ)) == Fraction(d(a, b), 3)
            for e in range(3):
                assert sum(w[q] * c[q][a] * c[q][b] * c[q][e] for q in range(NQ)) == 0
                for g in range(3):
                    iso = Fraction(d(a, b) * d(e, g) + d(a, e) * d(b, g) + d(a, g) * d(b, e), 9)
                    assert sum(w[q] * c[q][a] * c[q][b] * c[q][e] * c[q][g]
                               for q in range(NQ)) == iso


def test_p1_opposites():
    for q in range(NQ):
        assert OPP[OPP[q]] == q
        assert np.array_equal(C[OPP[q]], -C[q])
        assert WT[OPP[q]] == WT[q]


# ------------------------------------------------------------------ P2 rest state
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p2_rest_state_is_bitwise_invariant(seed):
    wl = W.random_mask((9, 8, 7), p_fluid=0.55, n_iolets=2, seed=seed)
    o = oracle.Oracle(wl.site_type, 0, 0.7, [1.0, 1.0])     # iolets at rho = 1: still at rest
    o.step(40)
    rho, u = o.get_macroscopic()
    assert np.all(rho == 1.0)
    assert np.all(u == 0.0)


# ------------------------------------------------------------------ P3 uniform flow
def test_p3_uniform_flow_is_a_fixed_point():
    st = np.ones((5, 6, 7), dtype=np.uint8)
    o = oracle.Oracle(st, 7, 0.83, [])
    n = o.n_sites
    rho0 = np.full(n, 1.03)
    u0 = np.tile(np.array([0.02, -0.01, 0.03]), (n, 1))
    o.set_state(rho0, u0)
    o.step(25)
    rho, u = o.get_macroscopic()
    assert np.max(np.abs(rho - 1.03)) < 1e-15
    assert np.max(np.abs(u - u0)) < 1e-16


# ------------------------------------------------------------------ P4/P5 conservation
def test_p4_p5_mass_and_momentum_conserved_periodic():
    wl = W.random_mask((8, 7, 6), p_fluid=1.1, n_iolets=0, periodic=7, seed=5)
    o = oracle.Oracle(wl.site_type, 7, 0.62, [])
    o.set_state(wl.rho0, wl.u0)
    r0, u0 = o.get_macroscopic()
    m0, j0 = r0.sum(), (r0[:, None] * u0).sum(axis=0)
    o.step(200)
    r1, u1 = o.get_macroscopic()
    assert abs(r1.sum() - m0) / o.n_sites < 1e-15
    assert np.max(np.abs((r1[:, None] * u1).sum(axis=0) - j0)) / o.n_sites < 1e-16
    assert np.max(np.abs(u1 - u0)) > 1e-4        # something did happen


def test_p4_mass_conserved_with_walls():
    wl = W.random_mask((9, 8, 7), p_fluid=0.6, n_iolets=0, periodic=2, seed=11)
    o = oracle.Oracle(wl.site_type, 2, 0.9, [])
    o.set_state(wl.rho0, wl.u0)
    m0 = o.get_macroscopic()[0].sum()
    o.step(150)
    assert abs(o.get_macroscopic()[0].sum() - m0) / o.n_sites < 1e-15


# ------------------------------------------------------------------ pure streaming
@pytest.mark.parametrize("q", range(19))
def test_streaming_moves_a_marked_population_along_c(q):
    if q >= NQ:
        pytest.skip("D3Q15 has 15 directions")
    """tau = 1e30 switches collision off (f* = f exactly in fp64); a marked population in
    slot q at x0 must be found in slot q at x0 + n c_q (periodic wrap) and nowhere else."""
    nx, ny, nz = 5, 4, 3
    st = np.ones((nz, ny, nx), dtype=np.uint8)
    o = oracle.Oracle(st, 7, 1e30, [])
    f = np.tile(WT, (o.n_sites, 1))
    x0 = (1, 2, 0)
    i0 = (x0[2] * ny + x0[1]) * nx + x0[0]
    f[i0, q] += 0.125
    o.set_populations(f)
    n = 7
    o.step(n)
    g = o.get_populations()
    x1 = ((x0[0] + n * C[q][0]) % nx, (x0[1] + n * C[q][1]) % ny, (x0[2] + n * C[q][2]) % nz)
    i1 = (x1[2] * ny + x1[1]) * nx + x1[0]
    expect = np.tile(WT, (o.n_sites, 1))
    expect[i1, q] += 0.125
    assert np.array_equal(g, expect)


def test_streaming_bounces_back_half_way():
    """1-D channel x = 0..3, outside solid: a population moving +x from x = 1 is at x = 2,
    x = 3 after 1, 2 steps, then reversed in the opposite slot at x = 3 (the wall sits
    half a link beyond x = 3), then at x = 2 moving -x."""
    st = np.ones((1, 1, 4), dtype=np.uint8)
    o = oracle.Oracle(st, 0, 1e30, [])
    qp = [q for q in range(NQ) if tuple(C[q]) == (1, 0, 0)][0]
    qm = OPP[qp]
    base = np.tile(WT, (4, 1))
    # y/z links all bounce back onto the same site, so the base state is stationary
    f = base.copy()
    f[1, qp] += 0.25
    o.set_populations(f)
    where = []
    for _ in range(5):
        o.step(1)
        d = o.get_populations() - base
        (i,), (q,) = np.nonzero(d)[0], np.nonzero(d)[1]
        assert d[i, q] == 0.25
        where.append((int(i), int(q)))
    assert where == [(2, qp), (3, qp), (3, qm), (2, qm), (1, qm)]


# ------------------------------------------------------------------ relaxation rate
@pytest.mark.parametrize("tau", [0.6, 1.0, 1.7])
def test_non_equilibrium_part_decays_by_one_minus_one_over_tau(tau):
    """1x1x1 periodic box: every neighbour is the site itself, so streaming is the identity
    and a mass- and momentum-free perturbation decays exactly as (1 - 1/tau)^n."""
    st = np.ones((1, 1, 1), dtype=np.uint8)
    o = oracle.Oracle(st, 7, tau, [])
    qx = [q for q in range(NQ) if tuple(C[q]) == (1, 0, 0)][0]
    q0 = [q for q in range(NQ) if tuple(C[q]) == (0, 0, 0)][0]
    pert = np.zeros(NQ)
    pert[qx] = pert[OPP[qx]] = 1e-3
    pert[q0] = -2e-3
    o.set_populations((WT + pert)[None, :])
    n = 9
    o.step(n)
    got = o.get_populations()[0] - WT
    assert np.max(np.abs(got - (1.0 - 1.0 / tau) ** n * pert)) < 1e-16   # ulp(w_0) = 2.8e-17


# ------------------------------------------------------------------ P6 shear wave
@pytest.mark.parametrize("tau", [0.6, 0.8, 1.2])
def test_p6_shear_wave_decays_at_nu(tau):
    ny = 64
    st = np.ones((1, ny, 1), dtype=np.uint8)
    o = oracle.Oracle(st, 7, tau, [])
    k = 2 * math.pi / ny
    u0 = np.zeros((ny, 3))
    u0[:, 0] = 1e-3 * np.sin(k * np.arange(ny))
    o.set_state(np.ones(ny), u0)
    T = 300
    o.step(T)
    _, u = o.get_macroscopic()
    amp = 2.0 / ny * np.dot(u[:, 0], np.sin(k * np.arange(ny)))
    nu = (tau - 0.5) / 3.0
    assert amp / 1e-3 == pytest.approx(math.exp(-nu * k * k * T), rel=4e-3)
    assert np.max(np.abs(u[:, 1:])) < 1e-15


# ------------------------------------------------------------------ P7 Taylor-Green
def test_p7_taylor_green_kinetic_energy_decay():
    wl = W.periodic_cube(n=32, tau=0.6, u0=0.01, nz=1)
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, [])
    o.set_state(wl.rho0, wl.u0)
    ke = []
    for _ in range(4):
        r, u = o.get_macroscopic()
        ke.append(0.5 * np.sum(r[:, None] * u * u))
        o.step(100)
    nu, k = (0.6 - 0.5) / 3.0, wl.info["k"]
    expect = math.exp(-4.0 * nu * k * k * 100)          # KE ~ exp(-4 nu k^2 t)
    for a, b in zip(ke[1:-1], ke[2:]):                   # skip the first (acoustic transient)
        assert b / a == pytest.approx(expect, rel=1e-3)
    assert ke[1] / ke[0] == pytest.approx(expect, rel=2e-2)   # start-up transient (rho = 1, f = feq)


# ------------------------------------------------------------------ P8 Poiseuille
@pytest.mark.parametrize("tau", [0.5 + math.sqrt(3.0 / 16.0), 0.9, 0.6])
def test_p8_plane_poiseuille_between_bounce_back_walls(tau):
    """Channel of H fluid rows between solid rows, periodic in x, density iolets in z.
    LBGK with halfway bounce-back has a closed-form steady solution (He, Zou, Luo & Dembo
    1997): the walls sit at y = 1/2 and y = H + 1/2 and the parabola carries a uniform
    numerical slip,
        u_z(y) = G/(2 nu) [ (y - 1/2)(H + 1/2 - y) + (16 (tau - 1/2)^2 - 3) / 12 ],
    which vanishes at tau = 1/2 + sqrt(3/16). G = -(1/3) d rho/dz is measured on the
    developed mid-section (the iolet rule A6 has an entrance layer, so the nominal
    (rho_in - rho_out)/(3L) is only approached to 7-25 %)."""
    H, L = 11, 24
    st = np.zeros((L + 2, H + 2, 1), dtype=np.uint8)
    st[1:L + 1, 1:H + 1, 0] = 1
    st[0, 1:H + 1, 0] = 2
    st[L + 1, 1:H + 1, 0] = 3
    o = oracle.Oracle(st, 1, tau, [1.0005, 0.9995], threads=4)
    o.step(8000)
    rho, u = o.get_macroscopic()
    x, y, z = canon_coords(st)
    za, zb = 9, 16
    G = (rho[z == za].mean() - rho[z == zb].mean()) / (3.0 * (zb - za))
    nu = (tau - 0.5) / 3.0
    assert G == pytest.approx(0.001 / (3.0 * L), rel=0.30) and G > 0      # flows inlet -> outlet
    mid = z == (L // 2)
    yy = y[mid].astype(float)
    slip = (16.0 * (tau - 0.5) ** 2 - 3.0) / 12.0
    expect = G / (2.0 * nu) * ((yy - 0.5) * (H + 0.5 - yy) + slip)
    got = (rho * u[:, 2])[mid]
    assert np.max(np.abs(got / expect - 1.0)) < 2.5e-3
    assert np.max(np.abs(u[mid, 0])) < 1e-12 and np.max(np.abs(u[mid, 1])) < 1e-5


def test_p8_pipe_poiseuille_config0():
    """BASELINE configs[0] geometry run to steady state (200 steps is not
    steady). u_max = G R^2 / (4 nu) = 1.6667e-3; staircase wall => loose tolerances."""
    wl = W.pipe()
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, threads=4)
    o.step(2500)
    rho, u = o.get_macroscopic()
    x, y, z = canon_coords(wl.site_type)
    R, L, nu = 8.0, 64.0, (wl.tau - 0.5) / 3.0
    G = (wl.iolet_rho[0] - wl.iolet_rho[1]) / (3.0 * L)
    umax = G * R * R / (4.0 * nu)
    centre = (z == 32) & (x == 8) & (y == 8)
    assert u[centre, 2][0] == pytest.approx(umax, rel=0.02)
    line = (z == 32) & (y == 8)
    r = np.abs(x[line] - 8.0)
    expect = G * (R * R - r * r) / (4.0 * nu)
    got = u[line, 2]
    assert np.linalg.norm(got - expect) / np.linalg.norm(expect) < 0.10
    assert np.max(np.abs(got - got[::-1])) < 1e-12                  # mirror symmetric
    assert np.all(got > 0)


# ------------------------------------------------------------------ Ladd velocity iolets
@pytest.mark.parametrize("tau", [0.6, 1.0, 1.4])
def test_ladd_moving_boundary_gives_exact_couette_flow(tau):
    """A velocity iolet is Ladd's bounce-back off a boundary moving with u_k (PAPER.md lines
    43, 59: "LADDIOLET"). Tangential motion above a channel of H rows whose lower wall is at
    rest: the steady state is plane Couette flow, which LBGK with halfway bounce-back
    represents exactly, u_x(y) = U (y - 1/2) / H with the walls at y = 1/2 and y = H + 1/2.
    A wrong factor (2 w rho c.u / c_s^2 = 6 w rho c.u) or sign changes the slope."""
    H, U = 8, 0.01
    st = np.zeros((1, H + 2, 1), dtype=np.uint8)
    st[0, 1:H + 1, 0] = 1
    st[0, H + 1, 0] = 2
    o = oracle.Oracle(st, 5, tau, [1.0])
    o.set_iolet_velocity([1], [[U, 0.0, 0.0]])
    o.step(int(40 * H * H / ((tau - 0.5) / 3.0) / 10))
    rho, u = o.get_macroscopic()
    y = np.arange(1, H + 1)
    assert np.max(np.abs(u[:, 0] - U * (y - 0.5) / H)) < 1e-13
    assert np.max(np.abs(u[:, 1:])) < 1e-16 and np.max(np.abs(rho - 1.0)) < 1e-15


def test_ladd_normal_inflow_injects_mass_flux_rho_times_u():
    """Normal motion: per step the boundary injects sum_q 6 w_q rho (c_q.u) over the links
    that cross it = rho u_n exactly (sum over c_qn = +1 of w_q c_qn^2 = 1/6). In a duct that is
    periodic sideways with a velocity inlet at one end and a constant-density outlet at the
    other, the steady mass flux is therefore rho(first site) * W everywhere."""
    L, Wn = 16, 0.005
    st = np.zeros((L + 2, 1, 1), dtype=np.uint8)
    st[1:L + 1, 0, 0] = 1
    st[0, 0, 0] = 2
    st[L + 1, 0, 0] = 3
    o = oracle.Oracle(st, 3, 0.8, [1.0, 1.0])
    o.set_iolet_velocity([1, 0], [[0.0, 0.0, Wn], [0.0, 0.0, 0.0]])
    o.step(40000)
    rho, u = o.get_macroscopic()
    j = rho * u[:, 2]
    assert np.max(np.abs(j - rho[0] * Wn)) < 1e-13
    assert np.max(np.abs(u[:, :2])) < 1e-16


def test_ladd_velocity_at_rest_is_plain_bounce_back():
    """u_k = 0 must reproduce a solid wall bit for bit."""
    wl = W.random_mask((8, 7, 6), p_fluid=0.6, n_iolets=2, p_iolet=0.1, seed=21)
    as_wall = wl.site_type.copy()
    as_wall[as_wall >= 2] = 0
    a = oracle.Oracle(wl.site_type, 0, wl.tau, wl.iolet_rho)
    a.set_iolet_velocity([1, 1], np.zeros((2, 3)))
    b = oracle.Oracle(as_wall, 0, wl.tau, [])
    for o in (a, b):
        o.set_state(wl.rho0, wl.u0)
        o.step(12)
    (ra, ua), (rb, ub) = a.get_macroscopic(), b.get_macroscopic()
    assert np.array_equal(ra, rb) and np.array_equal(ua, ub)


# ------------------------------------------------------------------ velocity weights (inlet profile)
def test_ladd_velocity_weights_special_cases():
    """Per-site weights omega(x) scale the prescribed velocity seen from site x (PAPER.md line
    59, USE_VELOCITY_WEIGHTS_FILE; reading R-weights): all ones is no weights, bit
    for bit; a uniform weight a is the iolet velocity a u_k; weight 0 everywhere is a wall."""
    wl = W.random_mask((9, 8, 7), p_fluid=0.65, n_iolets=2, p_iolet=0.1, periodic=2, seed=77)
    kind, u = [1, 0], np.array([[0.011, -0.004, 0.006], [0.0, 0.0, 0.0]])
    n = int(wl.n_sites)

    def run(weight, uk=u, st=wl.site_type, rho_io=wl.iolet_rho, kinds=kind):
        o = oracle.Oracle(st, 2, wl.tau, rho_io)
        o.set_state(wl.rho0, wl.u0)
        if kinds is not None:
            o.set_iolet_velocity(kinds, uk)
        o.set_iolet_weight(weight)
        o.step(15)
        return o.get_macroscopic()

    r0, u0 = run(None)
    r1, u1 = run(np.ones(n))
    assert np.array_equal(r0, r1) and np.array_equal(u0, u1)
    ra, ua = run(np.full(n, 0.37))
    rb, ub = run(None, uk=0.37 * u)
    assert np.max(np.abs(ra - rb)) < 1e-15 and np.max(np.abs(ua - ub)) < 1e-15
    assert np.max(np.abs(ua - u0)) > 1e-6                             # and it does matter
    rz, uz = run(np.zeros(n))                                         # boundary at rest = bounce-back
    rw, uw = run(None, uk=np.zeros((2, 3)))
    assert np.array_equal(rz, rw) and np.array_equal(uz, uw)


def test_ladd_velocity_weights_inject_the_weighted_mass_per_site(lattice):
    """One step from rest (rho = 1, u = 0, so f* = w): a site gains exactly
    sum over its velocity-iolet links q of 6 w_q omega(x) c_q.u_k, and nothing else moves mass.
    Evaluated voxel by voxel from the site types: pins which site's weight multiplies which
    link, the factor and the sign."""
    wl = W.random_mask((10, 9, 8), p_fluid=0.6, n_iolets=2, p_iolet=0.12, seed=5)
    st = wl.site_type
    nz, ny, nx = st.shape
    uk = np.array([[0.013, 0.007, -0.009], [-0.004, 0.01, 0.002]])
    rng = np.random.default_rng(3)
    om = rng.uniform(0.0, 2.0, int(wl.n_sites))
    o = oracle.Oracle(st, 0, 0.9, [1.0, 1.0])
    o.set_iolet_velocity([1, 1], uk)
    o.set_iolet_weight(om)
    o.step(1)
    rho, _ = o.get_macroscopic()
    c, w = C, WT                                                      # the lattice under test
    expect = np.zeros(int(wl.n_sites))
    for i, (x, y, z) in enumerate(zip(*canon_coords(st))):
        for q in range(len(w)):
            sx, sy, sz = x - c[q][0], y - c[q][1], z - c[q][2]
            if 0 <= sx < nx and 0 <= sy < ny and 0 <= sz < nz and st[sz, sy, sx] >= 2:
                k = int(st[sz, sy, sx]) - 2
                expect[i] += 6.0 * w[q] * om[i] * float(np.dot(c[q], uk[k]))
    assert np.max(np.abs(expect)) > 1e-3
    assert np.max(np.abs((rho - 1.0) - expect)) < 1e-15


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_ladd_velocity_weights_dense_twin(seed):
    """The dense push implementation carries the weights per voxel, independently."""
    wl = W.random_mask((8, 9, 7), p_fluid=0.65, n_iolets=3, p_iolet=0.09, periodic=seed, seed=700 + seed)
    st, vox = wl.site_type, wl.fluid_voxels()
    rng = np.random.default_rng(seed)
    kind, uio = np.array([1, 0, 1], dtype=np.uint8), 0.02 * (rng.random((3, 3)) - 0.5)
    om = rng.uniform(0.0, 2.0, len(vox))
    om_vox = np.zeros(st.size)
    om_vox[vox] = om
    rho0v, u0v = np.ones(st.size), np.zeros((st.size, 3))
    rho0v[vox], u0v[vox] = wl.rho0, wl.u0
    rd, ud = oracle.dense_run(st, seed, wl.tau, wl.iolet_rho, 11, rho0v, u0v, iolet_kind=kind, iolet_u=uio,
                              site_weight_vox=om_vox)
    o = oracle.Oracle(st, seed, wl.tau, wl.iolet_rho, variant=oracle.VARIANT_RAW)
    o.set_state(wl.rho0, wl.u0)
    o.set_iolet_velocity(kind, uio)
    o.set_iolet_weight(om)
    o.step(11)
    r, u = o.get_macroscopic()
    assert np.max(np.abs(r - rd.reshape(-1)[vox])) < 5e-15
    assert np.max(np.abs(u - ud.reshape(-1, 3)[vox])) < 5e-15
    o.set_iolet_weight(None)                                           # and the weights are not a no-op
    o.set_state(wl.rho0, wl.u0)
    o.step(11)
    assert np.max(np.abs(o.get_macroscopic()[1] - u)) > 1e-7


def test_inlet_profile_weights_average_to_one_and_vanish_at_the_rim():
    wl = W.with_inlet_profile(W.with_velocity_inlet(W.by_name("pipe")))
    w = wl.iolet_weight
    first = np.flatnonzero(w != 1.0)
    assert len(first) == 197                                           # the first slice of the pipe
    assert abs(w[first].mean() - 1.0) < 1e-12 and 1.7 < w[first].max() < 2.0 and 0.0 < w[first].min() < 0.25


# ------------------------------------------------------------------ normal-projected iolets
def test_iolet_normal_projection_special_cases():
    """(a) no normal, or a zero normal: unchanged bit for bit; (b) a flow that is exactly
    along the normal at the iolet sites (1-D duct): the projection changes nothing but
    roundoff; (c) a normal perpendicular to everything the iolet sites can do: the ghost is at
    rest, i.e. the rule becomes f_eq(rho_k, 0); (d) the length of the normal is irrelevant."""
    wl = W.random_mask((9, 8, 7), p_fluid=0.65, n_iolets=2, p_iolet=0.08, seed=12)

    def run(normals, st=wl.site_type, rho_io=wl.iolet_rho, steps=12):
        o = oracle.Oracle(st, 0, wl.tau, rho_io)
        if st is wl.site_type:
            o.set_state(wl.rho0, wl.u0)
        if normals is not None:
            o.set_iolet_normal(normals)
        o.step(steps)
        return o.get_populations()

    base = run(None)
    assert np.array_equal(base, run(np.zeros((2, 3))))
    proj = run([[1.0, 2.0, -1.0], [0.0, 0.0, 1.0]])
    assert np.max(np.abs(proj - base)) > 1e-6                       # it does something
    assert np.max(np.abs(proj - run([[3.0, 6.0, -3.0], [0.0, 0.0, 0.2]]))) < 1e-15   # (d)
    # (b), (c): a duct along z, periodic sideways
    L = 10
    st = np.zeros((L + 2, 1, 1), dtype=np.uint8)
    st[1:L + 1, 0, 0] = 1
    st[0, 0, 0], st[L + 1, 0, 0] = 2, 3
    rho_io = [1.002, 0.998]
    a = run(None, st, rho_io, 40)
    b = run([[0, 0, 1], [0, 0, -1]], st, rho_io, 40)
    assert np.max(np.abs(a - b)) < 1e-16
    c = run([[1, 0, 0], [0, 1, 0]], st, rho_io, 40)
    assert np.max(np.abs(a - c)) > 1e-7
    # ghost at rest: same as a run whose iolet sites see u = 0 in the rule -> compare with the
    # dense twin, which implements the projection independently
    rd, ud = oracle.dense_run(st, 3, wl.tau, rho_io, 40, iolet_normal=[[1, 0, 0], [0, 1, 0]])
    o = oracle.Oracle(st, 3, wl.tau, rho_io, variant=oracle.VARIANT_RAW)
    o.set_iolet_normal([[1, 0, 0], [0, 1, 0]])
    o.step(40)
    r, u = o.get_macroscopic()
    v = np.flatnonzero(st.reshape(-1) == 1)
    assert np.max(np.abs(r - rd.reshape(-1)[v])) < 1e-15 and np.max(np.abs(u - ud.reshape(-1, 3)[v])) < 1e-15


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_iolet_normal_projection_dense_twin(seed):
    wl = W.random_mask((8, 7, 9), p_fluid=0.65, n_iolets=3, p_iolet=0.08, periodic=seed, seed=600 + seed)
    st, vox = wl.site_type, wl.fluid_voxels()
    rng = np.random.default_rng(seed)
    normals = rng.standard_normal((3, 3))
    normals[1] = 0.0                                                  # one iolet without a normal
    kind, uio = np.array([0, 0, 1], dtype=np.uint8), 0.02 * (rng.random((3, 3)) - 0.5)
    rho0v, u0v = np.ones(st.size), np.zeros((st.size, 3))
    rho0v[vox], u0v[vox] = wl.rho0, wl.u0
    rd, ud = oracle.dense_run(st, seed, wl.tau, wl.iolet_rho, 9, rho0v, u0v, iolet_kind=kind, iolet_u=uio,
                              iolet_normal=normals)
    o = oracle.Oracle(st, seed, wl.tau, wl.iolet_rho, variant=oracle.VARIANT_RAW)
    o.set_state(wl.rho0, wl.u0)
    o.set_iolet_velocity(kind, uio)
    o.set_iolet_normal(normals)
    o.step(9)
    r, u = o.get_macroscopic()
    assert np.max(np.abs(r - rd.reshape(-1)[vox])) < 5e-15
    assert np.max(np.abs(u - ud.reshape(-1, 3)[vox])) < 5e-15


# ------------------------------------------------------------------ BFL interpolated walls
def _d27_index(dx, dy, dz):
    return (dz + 1) * 9 + (dy + 1) * 3 + (dx + 1)


@pytest.mark.parametrize("tau", [0.6, 1.0])
@pytest.mark.parametrize("d", [0.15, 0.5, 0.8, 1.0])
def test_bfl_wall_off_the_lattice_gives_exact_couette_flow(d, tau):
    """Interpolated bounce-back ("BFL", ref [16]): the lower wall sits
    the fraction d of a link below the first fluid row (at y = 1 - d, for every link that
    crosses it, axis or diagonal), the upper boundary is a Ladd wall moving with U at
    y = H + 1/2. Linear interpolation represents the linear Couette profile exactly:
    u_x(y) = U (y - y_w) / (H + 1/2 - y_w). Plain bounce-back would put the wall at y = 1/2."""
    H, U = 8, 0.01
    st = np.zeros((1, H + 2, 1), dtype=np.uint8)
    st[0, 1:H + 1, 0] = 1
    st[0, H + 1, 0] = 2
    o = oracle.Oracle(st, 5, tau, [1.0])
    o.set_iolet_velocity([1], [[U, 0.0, 0.0]])
    d27 = np.zeros((H, 27))
    for dz in (-1, 0, 1):
        for dx in (-1, 0, 1):
            d27[0, _d27_index(dx, -1, dz)] = d          # links of row y = 1 that point down
    o.set_wall_distance(d27)
    o.step(int(80 * H * H / ((tau - 0.5) / 3.0) / 10))
    _, u = o.get_macroscopic()
    y = np.arange(1, H + 1)
    yw = 1.0 - d
    assert np.max(np.abs(u[:, 0] - U * (y - yw) / (H + 0.5 - yw))) < 2e-12 * U / 0.01
    if d != 0.5:                                           # and it is not the halfway answer
        assert np.max(np.abs(u[:, 0] - U * (y - 0.5) / H)) > 1e-5


def test_bfl_at_half_a_link_is_plain_bounce_back_bitwise():
    wl = W.random_mask((9, 8, 7), p_fluid=0.6, n_iolets=2, p_iolet=0.06, periodic=1, seed=31)
    a = oracle.Oracle(wl.site_type, 1, wl.tau, wl.iolet_rho)
    b = oracle.Oracle(wl.site_type, 1, wl.tau, wl.iolet_rho)
    b.set_wall_distance(np.full((b.n_sites, 27), 0.5))
    for o in (a, b):
        o.set_state(wl.rho0, wl.u0)
        o.step(15)
    assert np.array_equal(a.get_populations(), b.get_populations())
    b.set_wall_distance(None)                               # switching it off again
    a.step(3)
    b.step(3)
    assert np.array_equal(a.get_populations(), b.get_populations())


@pytest.mark.parametrize("seed,periodic,shape", [(0, 0, (7, 6, 5)), (1, 7, (6, 6, 6)), (2, 1, (12, 5, 4)),
                                                 (3, 4, (5, 4, 11)), (4, 0, (12, 12, 12))])
def test_bfl_dense_push_twin_equals_sparse_pull(seed, periodic, shape):
    """The independently written dense push implementation, with random wall distances on
    every link (used only where the link is a wall link), velocity iolets mixed in."""
    wl = W.random_mask(shape, p_fluid=0.65, n_iolets=2, p_iolet=0.06, periodic=periodic,
                       tau=0.6 + 0.1 * seed, seed=400 + seed)
    st, vox = wl.site_type, wl.fluid_voxels()
    rng = np.random.default_rng(seed)
    d27 = rng.uniform(0.02, 1.0, size=(len(vox), 27))
    d27[rng.random(d27.shape) < 0.2] = 0.0                   # some links without a distance
    d27_vox = np.zeros((st.size, 27))
    d27_vox[vox] = d27
    rho0v, u0v = np.ones(st.size), np.zeros((st.size, 3))
    rho0v[vox], u0v[vox] = wl.rho0, wl.u0
    kind, uio = np.array([1, 0], dtype=np.uint8), 0.02 * (rng.random((2, 3)) - 0.5)
    steps = 10
    rd, ud = oracle.dense_run(st, periodic, wl.tau, wl.iolet_rho, steps, rho0v, u0v,
                              iolet_kind=kind, iolet_u=uio, wall_d27_vox=d27_vox)
    rd, ud = rd.reshape(-1)[vox], ud.reshape(-1, 3)[vox]
    o = oracle.Oracle(st, periodic, wl.tau, wl.iolet_rho, variant=oracle.VARIANT_RAW)
    o.set_state(wl.rho0, wl.u0)
    o.set_iolet_velocity(kind, uio)
    o.set_wall_distance(d27)
    o.step(steps)
    r, u = o.get_macroscopic()
    assert np.max(np.abs(r - rd)) < 5e-15 and np.max(np.abs(u - ud)) < 5e-15
    o2 = oracle.Oracle(st, periodic, wl.tau, wl.iolet_rho)    # without BFL it is another flow
    o2.set_state(wl.rho0, wl.u0)
    o2.set_iolet_velocity(kind, uio)
    o2.step(steps)
    assert np.max(np.abs(o2.get_macroscopic()[1] - u)) > 1e-6


# ------------------------------------------------------------------ viscous stress read-out
@pytest.mark.parametrize("tau", [0.6, 0.8, 1.4])
def test_stress_of_couette_flow_is_rho_nu_shear_rate(tau):
    """sigma_ab = -(1 - 1/(2 tau)) sum_q c_a c_b (f_q - f_eq_q). In steady plane Couette flow
    (exact in LBGK, see the Ladd pin) the shear stress is rho nu dU/dy at every site: pins the
    prefactor, the sign and the component order (xy is component 3)."""
    H, U = 8, 0.01
    st = np.zeros((1, H + 2, 1), dtype=np.uint8)
    st[0, 1:H + 1, 0] = 1
    st[0, H + 1, 0] = 2
    o = oracle.Oracle(st, 5, tau, [1.0])
    o.set_iolet_velocity([1], [[U, 0.0, 0.0]])
    o.step(int(60 * H * H / ((tau - 0.5) / 3.0) / 10))
    sg = o.get_stress()
    nu = (tau - 0.5) / 3.0
    assert sg.shape == (H, 6)
    assert np.max(np.abs(sg[:, 3] / (nu * U / H) - 1.0)) < 1e-11
    assert np.max(np.abs(sg[:, [4, 5]])) < 1e-18                     # no xz, yz shear
    assert np.max(np.abs(sg[:, :3])) < 10.0 * (U / H) ** 2           # normal stresses: O(shear^2)


def test_stress_of_poiseuille_flow_is_linear_and_balances_the_pressure_gradient():
    tau, H, L = 0.9, 11, 24
    st = np.zeros((L + 2, H + 2, 1), dtype=np.uint8)
    st[1:L + 1, 1:H + 1, 0] = 1
    st[0, 1:H + 1, 0] = 2
    st[L + 1, 1:H + 1, 0] = 3
    o = oracle.Oracle(st, 1, tau, [1.0005, 0.9995], threads=4)
    o.step(8000)
    rho, _ = o.get_macroscopic()
    sg = o.get_stress()
    x, y, z = canon_coords(st)
    G = (rho[z == 9].mean() - rho[z == 16].mean()) / (3.0 * 7)     # -dp/dz on the mid-section
    mid = z == 12
    yy = y[mid].astype(float)
    expect = -G * (yy - (H + 1) / 2.0)                             # momentum balance d sigma_yz/dy = -G
    got = sg[mid, 5]
    off = yy != (H + 1) / 2.0
    assert np.max(np.abs(got[off] / expect[off] - 1.0)) < 5e-3
    assert abs(got[~off][0]) < 1e-3 * np.max(np.abs(expect))         # zero on the centre line
    assert np.max(np.abs(got + got[::-1])) < 1e-12 * np.max(np.abs(got))   # antisymmetric


def test_wall_shear_stress_of_channel_flows():
    """Couette: the traction on a plane with normal y is (rho nu U/H, 0, 0), all of it
    tangential -> WSS = rho nu U / H at every site, 0 where no normal is given, and the same
    for any length or sign of the normal. A normal along the flow sees no shear in Couette
    flow up to the O(shear^2) normal stresses."""
    H, U, tau = 8, 0.01, 0.8
    st = np.zeros((1, H + 2, 1), dtype=np.uint8)
    st[0, 1:H + 1, 0] = 1
    st[0, H + 1, 0] = 2
    o = oracle.Oracle(st, 5, tau, [1.0])
    o.set_iolet_velocity([1], [[U, 0.0, 0.0]])
    o.step(20000)
    nu = (tau - 0.5) / 3.0
    normals = np.zeros((H, 3))
    normals[0] = (0.0, 1.0, 0.0)
    normals[-1] = (0.0, -3.0, 0.0)
    normals[3] = (0.0, 0.5, 0.0)
    wss = o.get_wall_shear_stress(normals)
    for i in (0, 3, H - 1):
        assert wss[i] == pytest.approx(nu * U / H, rel=1e-10)
    assert np.all(wss[[1, 2, 4, 5, 6]] == 0.0)
    tilted = np.tile(np.array([1.0, 1.0, 0.0]), (H, 1))      # 45 degrees: t = s (1,1)/sqrt2 + normal parts
    w45 = o.get_wall_shear_stress(tilted)
    sg = o.get_stress()
    n = np.array([1.0, 1.0, 0.0]) / math.sqrt(2.0)
    for i in range(H):
        S = np.array([[sg[i, 0], sg[i, 3], sg[i, 4]], [sg[i, 3], sg[i, 1], sg[i, 5]], [sg[i, 4], sg[i, 5], sg[i, 2]]])
        t = S @ n
        assert w45[i] == pytest.approx(np.linalg.norm(t - (t @ n) * n), rel=1e-12)


def test_stress_vanishes_at_equilibrium():
    st = np.ones((4, 5, 6), dtype=np.uint8)
    o = oracle.Oracle(st, 7, 0.7, [])
    n = o.n_sites
    o.set_state(np.full(n, 1.02), np.tile(np.array([0.03, -0.02, 0.01]), (n, 1)))
    assert np.max(np.abs(o.get_stress())) < 1e-17
    o.step(9)
    assert np.max(np.abs(o.get_stress())) < 1e-17


# ------------------------------------------------------------------ P9 dense twin
@pytest.mark.parametrize("seed,periodic,shape", [
    (0, 0, (7, 6, 5)), (1, 7, (6, 6, 6)), (2, 1, (12, 5, 4)), (3, 2, (4, 9, 5)),
    (4, 4, (5, 4, 11)), (5, 5, (8, 3, 7)), (6, 0, (12, 12, 12)), (7, 7, (1, 1, 3)),
    (8, 3, (2, 2, 2)),
])
def test_p9_dense_push_twin_equals_sparse_pull(seed, periodic, shape):
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=3, p_iolet=0.08, periodic=periodic,
                       tau=0.5 + 0.1 * (1 + seed), seed=100 + seed)
    steps = 12
    st = wl.site_type
    vox = wl.fluid_voxels()
    nvox = st.size
    rho0v = np.ones(nvox)
    u0v = np.zeros((nvox, 3))
    rho0v[vox] = wl.rho0
    u0v[vox] = wl.u0
    rng = np.random.default_rng(seed)
    for kind, uio in ((None, None),
                      (np.array([1, 0, 1], dtype=np.uint8), 0.02 * (rng.random((3, 3)) - 0.5))):
        rd, ud = oracle.dense_run(st, periodic, wl.tau, wl.iolet_rho, steps, rho0v, u0v,
                                  iolet_kind=kind, iolet_u=uio)
        rd, ud = rd.reshape(-1)[vox], ud.reshape(-1, 3)[vox]
        for variant, tol in ((oracle.VARIANT_RAW, 2e-15), (oracle.VARIANT_SHIFTED, 2e-14)):
            o = oracle.Oracle(st, periodic, wl.tau, wl.iolet_rho, variant=variant)
            assert np.array_equal(o.site_voxels(), vox)
            o.set_state(wl.rho0, wl.u0)
            if kind is not None:
                o.set_iolet_velocity(kind, uio)
            o.step(steps)
            r, u = o.get_macroscopic()
            assert np.max(np.abs(r - rd)) < tol
            assert np.max(np.abs(u - ud)) < tol


# ------------------------------------------------------------------ P11 symmetry
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p11_mirror_symmetry(axis):
    wl = W.random_mask((7, 6, 5), p_fluid=0.65, n_iolets=2, seed=42)
    st = wl.site_type
    np_axis = 2 - axis                     # array is [z, y, x]
    st_m = np.ascontiguousarray(np.flip(st, axis=np_axis))
    nz, ny, nx = st.shape
    # scatter canonical fields to voxel grids, flip, gather back in the mirrored canonical order
    vox = wl.fluid_voxels()
    rho_v = np.zeros(st.size)
    u_v = np.zeros((st.size, 3))
    rho_v[vox] = wl.rho0
    u_v[vox] = wl.u0
    rho_m = np.flip(rho_v.reshape(nz, ny, nx), axis=np_axis).reshape(-1)
    u_m = np.flip(u_v.reshape(nz, ny, nx, 3), axis=np_axis).reshape(-1, 3).copy()
    u_m[:, axis] *= -1.0
    vox_m = np.flatnonzero(st_m.reshape(-1) == 1)
    a = oracle.Oracle(st, 0, wl.tau, wl.iolet_rho)
    a.set_state(wl.rho0, wl.u0)
    b = oracle.Oracle(st_m, 0, wl.tau, wl.iolet_rho)
    b.set_state(rho_m[vox_m], u_m[vox_m])
    a.step(15)
    b.step(15)
    ra, ua = a.get_macroscopic()
    rb, ub = b.get_macroscopic()
    ra_v = np.zeros(st.size)
    ua_v = np.zeros((st.size, 3))
    ra_v[vox] = ra
    ua_v[vox] = ua
    ra_m = np.flip(ra_v.reshape(nz, ny, nx), axis=np_axis).reshape(-1)[vox_m]
    ua_m = np.flip(ua_v.reshape(nz, ny, nx, 3), axis=np_axis).reshape(-1, 3)[vox_m].copy()
    ua_m[:, axis] *= -1.0
    assert np.max(np.abs(rb - ra_m)) < 1e-15
    assert np.max(np.abs(ub - ua_m)) < 1e-16


def test_p11_axis_permutation_symmetry():
    """Swapping the x and z axes of geometry and state swaps them in the result."""
    wl = W.random_mask((6, 5, 4), p_fluid=0.7, n_iolets=1, seed=9)
    st = wl.site_type
    st_p = np.ascontiguousarray(st.transpose(2, 1, 0))          # [x, y, z] as new [z, y, x]
    vox = wl.fluid_voxels()
    nz, ny, nx = st.shape
    rho_v = np.zeros(st.size)
    u_v = np.zeros((st.size, 3))
    rho_v[vox] = wl.rho0
    u_v[vox] = wl.u0
    rho_p = rho_v.reshape(nz, ny, nx).transpose(2, 1, 0).reshape(-1)
    u_p = u_v.reshape(nz, ny, nx, 3).transpose(2, 1, 0, 3).reshape(-1, 3)[:, ::-1]
    vox_p = np.flatnonzero(st_p.reshape(-1) == 1)
    a = oracle.Oracle(st, 0, wl.tau, wl.iolet_rho)
    a.set_state(wl.rho0, wl.u0)
    b = oracle.Oracle(st_p, 0, wl.tau, wl.iolet_rho)
    b.set_state(rho_p[vox_p], np.ascontiguousarray(u_p[vox_p]))
    a.step(10)
    b.step(10)
    ra, ua = a.get_macroscopic()
    rb, ub = b.get_macroscopic()
    ra_v = np.zeros(st.size)
    ua_v = np.zeros((st.size, 3))
    ra_v[vox] = ra
    ua_v[vox] = ua
    ra_p = ra_v.reshape(nz, ny, nx).transpose(2, 1, 0).reshape(-1)[vox_p]
    ua_p = ua_v.reshape(nz, ny, nx, 3).transpose(2, 1, 0, 3).reshape(-1, 3)[vox_p][:, ::-1]
    assert np.max(np.abs(rb - ra_p)) < 1e-15
    assert np.max(np.abs(ub - ua_p)) < 1e-16


# ------------------------------------------------------------------ P12 roundoff yardstick
def test_p12_long_double_twin_bounds_the_oracles_roundoff():
    wl = W.periodic_cube(n=16, tau=0.6, u0=0.01, nz=2)
    res = {}
    for v in (oracle.VARIANT_SHIFTED, oracle.VARIANT_RAW, oracle.VARIANT_SHIFTED_LD,
              oracle.VARIANT_RAW_LD):
        o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, [], variant=v)
        o.set_state(wl.rho0, wl.u0)
        o.step(300)
        res[v] = o.get_macroscopic()
    ref_r, ref_u = res[oracle.VARIANT_SHIFTED_LD]
    umax = np.max(np.linalg.norm(ref_u, axis=1))

    def err(v):
        r, u = res[v]
        return np.max(np.abs(r - ref_r)), np.max(np.abs(u - ref_u)) / umax

    e_rho, e_u = err(oracle.VARIANT_SHIFTED)
    assert e_rho < 1e-15 and e_u < 5e-14          # the oracle: orders below the 1e-12 budget
    e_rho, e_u = err(oracle.VARIANT_RAW)
    assert e_rho < 1e-13 and e_u < 1e-11          # raw f: same iteration, roundoff near 1e-12
    e_rho, e_u = err(oracle.VARIANT_RAW_LD)
    assert e_rho < 1e-15 and e_u < 1e-13


# ------------------------------------------------------------------ degenerate cases
def test_isolated_site_and_argument_checks():
    st = np.zeros((3, 3, 3), dtype=np.uint8)
    st[1, 1, 1] = 1
    o = oracle.Oracle(st, 0, 0.8, [])
    o.set_state(np.array([1.01]), np.array([[0.01, 0.0, 0.0]]))
    o.step(5)
    rho, u = o.get_macroscopic()
    assert rho[0] == pytest.approx(1.01, abs=1e-15)          # mass stays on the site
    with pytest.raises(ValueError):
        oracle.Oracle(st, 0, 0.5, [])                         # tau must exceed 1/2
    st[0, 0, 0] = 4
    with pytest.raises(ValueError):
        oracle.Oracle(st, 0, 0.8, [1.0])                      # type 4 needs 3 iolets
