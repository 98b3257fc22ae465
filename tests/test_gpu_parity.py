"""GPU parity: the CUDA path (through the C-ABI binding) against the oracle, element by
element, on the same seeded inputs.

Bar (BASELINE.json north_star): fp64 rho and u within 1e-12 relative max error, the
fp32-storage variant within 1e-5. Norm (reading R-norm):
E_rho = max|rho - rho_ref| / max|rho_ref|,  E_u = max_{x,a}|u_a - u_ref,a| / max_x |u_ref|_2.
"""
import dataclasses
import math
import os

import numpy as np
import pytest

import oracle
import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def hlb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1906_11925_b200 as m
    return m


def flags_of(hlb, scheme, store, order="morton", links="auto", lattice="d3q15", resident=False):
    """resident=False: the tests' small geometries would otherwise all take the resident
    multi-step kernel (hlb_step, include/hlb.h) instead of the one-shot step kernels the large
    configs run; the resident kernel has its own tests below."""
    f = hlb.HLB_AA if scheme == "aa" else hlb.HLB_TWO_LATTICE
    f |= 0 if resident else hlb.HLB_NO_RESIDENT
    f |= hlb.HLB_STORE_F32 if store == "f32" else hlb.HLB_STORE_F64
    f |= {"auto": hlb.HLB_ORDER_AUTO, "morton": hlb.HLB_ORDER_MORTON, "raster": hlb.HLB_ORDER_RASTER,
          "tiled": hlb.HLB_ORDER_TILED}[order]
    f |= {"auto": hlb.HLB_LINKS_AUTO, "table": hlb.HLB_LINKS_TABLE, "records": hlb.HLB_LINKS_RECORDS}[links]
    f |= {"d3q15": hlb.HLB_LATTICE_D3Q15, "d3q19": hlb.HLB_LATTICE_D3Q19}[lattice]
    return f


def errors(rho, u, rho_ref, u_ref):
    e_rho = np.max(np.abs(rho - rho_ref)) / np.max(np.abs(rho_ref))
    un = np.max(np.linalg.norm(u_ref, axis=1))
    e_u = np.max(np.abs(u - u_ref)) / (un if un > 0 else 1.0)
    return e_rho, e_u


def run_gpu(hlb, wl, steps, scheme, store, order="morton", links="auto", lattice="d3q15", extra=0):
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, store, order, links, lattice) | extra)
    assert g.hlb_num_q() == {"d3q15": 15, "d3q19": 19}[lattice]
    if links != "auto":
        assert g.hlb_uses_records() == (links == "records")
    if wl.rho0 is not None or wl.u0 is not None:
        g.hlb_set_state(wl.rho0, wl.u0)
    if wl.iolet_kind is not None:
        g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
    if wl.iolet_normal is not None:
        g.hlb_set_iolet_normal(wl.iolet_normal)
    if wl.iolet_weight is not None:
        g.hlb_set_iolet_weight(wl.iolet_weight)
    if wl.wall_distance is not None:
        g.hlb_set_wall_distance(wl.wall_distance)
        assert g.hlb_num_bfl_sites() > 0
    g.hlb_step(steps)
    assert g.hlb_steps_done() == steps
    out = g.hlb_get_macroscopic()
    g.close()
    return out


def run_oracle(wl, steps, threads=0, lattice="d3q15"):
    return oracle.run(wl, steps=steps, threads=threads, lattice=lattice)


_oracle_cache = {}


def oracle_cached(name, steps, lattice="d3q15"):
    key = (name, steps, lattice)
    if key not in _oracle_cache:
        _oracle_cache[key] = run_oracle(W.by_name(name, small=True), steps, lattice=lattice)
    return _oracle_cache[key]


# ------------------------------------------------------------- the five configs, scaled down
@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("name", W.CONFIG_NAMES)
def test_small_configs_match_oracle(hlb, name, scheme, store):
    wl = W.by_name(name, small=True)
    for steps in (wl.steps, wl.steps + 1):            # even and odd (A-A read-out parity)
        rho_ref, u_ref = oracle_cached(name, steps)
        rho, u = run_gpu(hlb, wl, steps, scheme, store)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)


@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("name", W.CONFIG_NAMES)
def test_small_configs_match_oracle_through_link_records(hlb, name, scheme, store):
    """The run-length link records (the form the step kernels read on x-fastest orders)
    against the oracle, raster order, records forced."""
    wl = W.by_name(name, small=True)
    steps = wl.steps + 1
    rho_ref, u_ref = oracle_cached(name, steps)
    rho, u = run_gpu(hlb, wl, steps, scheme, store, "raster", "records")
    e_rho, e_u = errors(rho, u, rho_ref, u_ref)
    assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)


@pytest.mark.parametrize("order", ["morton", "raster", "tiled"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_link_records_and_table_agree_bitwise(hlb, scheme, order):
    """Records and table describe the same links: bitwise identical results, whatever the
    share of sentinel records (morton: nearly all; raster: few)."""
    for name, steps in (("aneurysm", 33), ("cube", 12)):
        wl = W.by_name(name, small=True)
        a = run_gpu(hlb, wl, steps, scheme, "f64", order, "table")
        b = run_gpu(hlb, wl, steps, scheme, "f64", order, "records")
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


@pytest.mark.parametrize("order", ["raster", "tiled"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_result_is_independent_of_site_order(hlb, scheme, order):
    """P10: the internal order never leaks -- bitwise identical canonical results."""
    wl = W.by_name("aneurysm", small=True)
    a = run_gpu(hlb, wl, 41, scheme, "f64", "morton")
    b = run_gpu(hlb, wl, 41, scheme, "f64", order)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


@pytest.mark.parametrize("store", ["f64", "f32"])
def test_aa_equals_two_lattice_bitwise(hlb, store):
    """P14: same per-site arithmetic, so the two schemes agree bit for bit."""
    wl = W.by_name("tree", small=True)
    for steps in (6, 7):
        a = run_gpu(hlb, wl, steps, "two_lattice", store)
        b = run_gpu(hlb, wl, steps, "aa", store)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


# ------------------------------------------------------------- D3Q19
@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("name", W.CONFIG_NAMES)
def test_d3q19_small_configs_match_oracle(hlb, name, scheme, store):
    """The lattice the paper names: same five geometries, same
    tolerances, table links at an even and record links at an odd step count."""
    wl = W.by_name(name, small=True)
    for steps, order, links in ((wl.steps, "morton", "table"), (wl.steps + 1, "raster", "records")):
        rho_ref, u_ref = oracle_cached(name, steps, "d3q19")
        rho, u = run_gpu(hlb, wl, steps, scheme, store, order, links, "d3q19")
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)


def test_d3q19_differs_from_d3q15(hlb):
    """Guard against a lattice flag that is silently ignored."""
    wl = W.by_name("aneurysm", small=True)
    a = run_gpu(hlb, wl, 30, "two_lattice", "f64", "raster", "auto", "d3q15")
    b = run_gpu(hlb, wl, 30, "two_lattice", "f64", "raster", "auto", "d3q19")
    assert np.max(np.abs(a[1] - b[1])) > 1e-8


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_d3q19_variants_agree_bitwise(hlb, scheme):
    """D3Q19: records = table, every site order, 64-bit offsets, no prefetch, no graph, and
    A-A = two-lattice -- all bitwise."""
    wl = W.by_name("tree", small=True)
    steps = 35
    ref = run_gpu(hlb, wl, steps, scheme, "f64", "raster", "table", "d3q19")
    for order, links, extra in (("raster", "records", 0), ("morton", "records", 0),
                                ("tiled", "table", 0), ("raster", "records", hlb.HLB_INDEX64),
                                ("raster", "records", hlb.HLB_NO_PREFETCH | hlb.HLB_NO_GRAPH),
                                ("raster", "records", hlb.HLB_NO_PDL), ("morton", "table", hlb.HLB_NO_PDL)):
        got = run_gpu(hlb, wl, steps, scheme, "f64", order, links, "d3q19", extra)
        assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1]), (order, links, extra)
    other = run_gpu(hlb, wl, steps, "aa" if scheme == "two_lattice" else "two_lattice", "f64",
                    "raster", "records", "d3q19")
    assert np.array_equal(ref[0], other[0]) and np.array_equal(ref[1], other[1])


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("seed,periodic,shape", [
    (0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (33, 5, 4)), (5, 7, (1, 1, 3)), (7, 0, (24, 20, 18)),
    (8, 5, (40, 9, 23)),
])
def test_d3q19_random_masks_match_oracle(hlb, scheme, seed, periodic, shape):
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=3, p_iolet=0.06, periodic=periodic,
                       tau=0.55 + 0.07 * seed, seed=300 + seed)
    links, order = ("records", "raster") if seed % 2 else ("table", "morton")
    for steps in (0, 1, 2, 9, 10):
        rho_ref, u_ref = run_oracle(wl, steps, threads=1, lattice="d3q19")
        rho, u = run_gpu(hlb, wl, steps, scheme, "f64", order, links, "d3q19")
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < 1e-13 and e_u < 1e-12, (steps, e_rho, e_u)


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_d3q19_populations_match_oracle(hlb, scheme):
    wl = W.random_mask((12, 11, 10), p_fluid=0.65, n_iolets=2, periodic=1, tau=0.7, seed=78)
    c_o = oracle.velocity_set("d3q19")[0]
    c_g = hlb.hlb_lattice(hlb.HLB_LATTICE_D3Q19)[0]
    perm = [int(np.flatnonzero((c_g == c).all(axis=1))[0]) for c in c_o]     # oracle q -> library q
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, lattice="d3q19")
    o.set_state(wl.rho0, wl.u0)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, "f64", "raster", "auto", "d3q19"))
    g.hlb_set_state(wl.rho0, wl.u0)
    for steps in (0, 1, 4, 3):
        o.step(steps)
        g.hlb_step(steps)
        fo, fg = o.get_populations(), g.hlb_get_populations()
        assert fg.shape == fo.shape == (wl.n_sites, 19)
        assert np.max(np.abs(fg[:, perm] - fo)) < 1e-15
    fo = o.get_populations()
    fg = np.empty_like(fo)
    fg[:, perm] = fo
    g.hlb_set_populations(fg)
    o.step(5)
    g.hlb_step(5)
    assert np.max(np.abs(g.hlb_get_populations()[:, perm] - o.get_populations())) < 1e-15
    g.close()


# ------------------------------------------------------------- Ladd velocity iolets (NEXT-2)
@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("name", ["pipe", "aneurysm", "tree"])
def test_velocity_inlet_matches_oracle(hlb, name, scheme, lattice):
    """The paper's boundary set: Ladd velocity inlet + constant-density
    outlets, both storage types, even and odd step counts."""
    wl = W.with_velocity_inlet(W.by_name(name, small=True))
    for steps, store, order, links in ((wl.steps, "f64", "raster", "records"),
                                       (wl.steps + 1, "f64", "morton", "table"),
                                       (wl.steps + 1, "f32", "raster", "auto")):
        rho_ref, u_ref = run_oracle(wl, steps, lattice=lattice)
        rho, u = run_gpu(hlb, wl, steps, scheme, store, order, links, lattice)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)
    assert np.max(np.abs(u_ref)) > 1e-4                     # the inlet does drive a flow


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_time_varying_velocity_inlet_and_mixed_kinds(hlb, scheme):
    """A pulsatile inlet (the paper drives its inlet with a velocity waveform, Fig. 8): the
    velocity changes between hlb_step calls; random masks mix walls, density and velocity
    iolets on one site. Also switching an iolet back to the density rule."""
    wl = W.random_mask((14, 12, 10), p_fluid=0.65, n_iolets=3, p_iolet=0.07, periodic=2, tau=0.62,
                       seed=91)
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, "f64", "raster", "auto"))
    o.set_state(wl.rho0, wl.u0)
    g.hlb_set_state(wl.rho0, wl.u0)
    rng = np.random.default_rng(4)
    for it in range(6):
        kind = np.array([1, it % 2, 1 - it % 2], dtype=np.uint8)
        u = 0.02 * math.sin(0.9 * it + 0.3) * (rng.random((3, 3)) - 0.5)
        o.set_iolet_velocity(kind, u)
        g.hlb_set_iolet_velocity(kind, u)
        n = 3 + it
        o.step(n)
        g.hlb_step(n)
        e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o.get_macroscopic())
        assert e_rho < 1e-13 and e_u < 1e-12, (it, e_rho, e_u)
    g.hlb_set_iolet_velocity(None, None)                    # all back to constant density
    g.hlb_set_iolet_density([1.01, 0.99, 1.0])
    o2 = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, [1.01, 0.99, 1.0])
    o2.set_populations(o.get_populations())
    o2.step(7)
    g.hlb_step(7)
    e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o2.get_macroscopic())
    assert e_rho < 1e-13 and e_u < 1e-12
    with pytest.raises(hlb.HlbError):
        g.hlb_set_iolet_velocity([2, 0, 0], np.zeros((3, 3)))
    g.close()


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_velocity_inlet_with_profile_matches_oracle(hlb, scheme, lattice):
    """Per-site velocity weights (the paper's USE_VELOCITY_WEIGHTS_FILE flag):
    a parabolic profile across the inlet cap, in every site order (the weights cross the
    boundary in canonical order), both storage types, even and odd step counts; also through
    the resident multi-step kernel, and random weights on random masks with mixed iolet kinds."""
    for name in ("pipe", "aneurysm", "tree"):
        wl = W.with_inlet_profile(W.with_velocity_inlet(W.by_name(name, small=True)))
        for steps, store, order, links in ((wl.steps, "f64", "raster", "records"),
                                           (wl.steps + 1, "f64", "morton", "table"),
                                           (wl.steps + 1, "f32", "tiled", "auto")):
            rho_ref, u_ref = run_oracle(wl, steps, lattice=lattice)
            rho, u = run_gpu(hlb, wl, steps, scheme, store, order, links, lattice)
            e_rho, e_u = errors(rho, u, rho_ref, u_ref)
            assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)
        plain = run_oracle(W.with_velocity_inlet(W.by_name(name, small=True)), wl.steps, lattice=lattice)
        assert np.max(np.abs(plain[1] - run_oracle(wl, wl.steps, lattice=lattice)[1])) > 1e-6  # it matters
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                    flags_of(hlb, scheme, "f64", "raster", "auto", lattice, resident=True))
        g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
        g.hlb_set_iolet_weight(wl.iolet_weight)
        g.hlb_step(wl.steps)
        assert g.hlb_launch_count() == 1
        e_rho, e_u = errors(*g.hlb_get_macroscopic(), *run_oracle(wl, wl.steps, lattice=lattice))
        g.close()
        assert e_rho < 1e-12 and e_u < 1e-12, (name, "resident", e_rho, e_u)
    wl = W.random_mask((13, 12, 11), p_fluid=0.65, n_iolets=3, p_iolet=0.08, periodic=1, tau=0.6, seed=123)
    rng = np.random.default_rng(9)
    kind, uio = np.array([1, 0, 1], dtype=np.uint8), 0.02 * (rng.random((3, 3)) - 0.5)
    om = rng.uniform(0.0, 2.0, int(wl.n_sites))
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, lattice=lattice)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, "f64", "morton", "auto", lattice))
    for x in (o, g):
        (x.set_state if x is o else x.hlb_set_state)(wl.rho0, wl.u0)
    o.set_iolet_velocity(kind, uio)
    o.set_iolet_weight(om)
    g.hlb_set_iolet_velocity(kind, uio)
    g.hlb_set_iolet_weight(om)
    o.step(9)
    g.hlb_step(9)
    e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o.get_macroscopic())
    assert e_rho < 1e-13 and e_u < 1e-12
    g.hlb_set_iolet_weight(None)                             # removed: omega = 1 again
    o.set_iolet_weight(None)
    o.step(6)
    g.hlb_step(6)
    e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o.get_macroscopic())
    assert e_rho < 1e-13 and e_u < 1e-12
    with pytest.raises(hlb.HlbError):
        g.hlb_set_iolet_weight(np.full(int(wl.n_sites), np.inf))
    g.close()


def _oracle_with_waveform(wl, wave, steps, lattice):
    """The definition the waveform must reproduce: the oracle stepped one time level at a time,
    its velocity iolets set to u[t mod n_t] before the step from t to t+1."""
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, lattice=lattice)
    if wl.rho0 is not None or wl.u0 is not None:
        o.set_state(wl.rho0, wl.u0)
    if wl.iolet_weight is not None:
        o.set_iolet_weight(wl.iolet_weight)
    for t in range(steps):
        o.set_iolet_velocity(wl.iolet_kind, wave[t % len(wave)])
        o.step(1)
    out = o.get_macroscopic()
    o.close()
    return out


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_inlet_waveform_matches_per_step_oracle(hlb, scheme, lattice):
    """Device-resident inlet waveform (the paper's inlet velocity file):
    hlb_step(n) over several periods, with a read-out in between, against the oracle driven one
    step at a time. 71 steps on a small geometry would use the 32-step graph replay if the
    waveform did not switch it off (a captured launch fixes its time level)."""
    for name, store, n_t, steps in (("pipe", "f64", 7, 71), ("aneurysm", "f64", 5, 18),
                                    ("tree", "f32", 9, 23)):
        wl = W.with_velocity_inlet(W.by_name(name, small=True))
        if name == "aneurysm":                                # waveform x inlet profile
            wl = W.with_inlet_profile(wl)
        wave = W.pulsatile_waveform(wl, n_t)
        rho_ref, u_ref = _oracle_with_waveform(wl, wave, steps, lattice)
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                    flags_of(hlb, scheme, store, "raster", "auto", lattice))
        g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
        g.hlb_set_iolet_waveform(wave)
        if wl.iolet_weight is not None:
            g.hlb_set_iolet_weight(wl.iolet_weight)
        launches0 = g.hlb_launch_count()
        g.hlb_step(n_t + 1)
        g.hlb_get_macroscopic()                               # a read-out in mid-period
        g.hlb_step(steps - n_t - 1)
        assert g.hlb_steps_done() == steps
        assert g.hlb_launch_count() - launches0 == steps      # one fused kernel per time level
        e_rho, e_u = errors(*g.hlb_get_macroscopic(), rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, lattice, e_rho, e_u)
        g.close()
        assert np.max(np.abs(u_ref)) > 1e-4


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_inlet_waveform_is_bitwise_the_host_driven_sequence(hlb, scheme):
    """The waveform is only another way of handing u_k(t) to the same kernels: populations are
    bitwise those of hlb_set_iolet_velocity before every step. Also: the time restarts with
    hlb_set_state, later density / kind changes keep the waveform, NULL removes it."""
    wl = W.random_mask((13, 11, 12), p_fluid=0.7, n_iolets=3, p_iolet=0.08, periodic=1, tau=0.58, seed=17)
    kind = np.array([1, 0, 1], dtype=np.uint8)
    rng = np.random.default_rng(5)
    n_t = 4
    wave = 0.02 * (rng.random((n_t, 3, 3)) - 0.5)
    flags = flags_of(hlb, scheme, "f64", "raster", "auto")
    a = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags)
    b = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags)
    for x in (a, b):
        x.hlb_set_state(wl.rho0, wl.u0)
    a.hlb_set_iolet_velocity(kind, np.zeros((3, 3)))
    a.hlb_set_iolet_waveform(wave)
    a.hlb_step(11)
    for t in range(11):
        b.hlb_set_iolet_velocity(kind, wave[t % n_t])
        b.hlb_step(1)
    assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations())
    # densities and kinds change, the waveform stays; time restarts at 0 with hlb_set_state
    rho2 = [1.004, 0.997, 1.001]
    kind2 = np.array([0, 1, 1], dtype=np.uint8)
    for x in (a, b):
        x.hlb_set_state(wl.rho0, wl.u0)
        x.hlb_set_iolet_density(rho2)
    a.hlb_set_iolet_velocity(kind2, np.zeros((3, 3)))
    a.hlb_step(6)
    for t in range(6):
        b.hlb_set_iolet_velocity(kind2, wave[t % n_t])
        b.hlb_step(1)
    assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations())
    # removed: back to the constant vectors
    const_u = 0.01 * (rng.random((3, 3)) - 0.5)
    a.hlb_set_iolet_waveform(None)
    a.hlb_set_iolet_velocity(kind2, const_u)
    b.hlb_set_iolet_velocity(kind2, const_u)
    a.hlb_step(5)
    b.hlb_step(5)
    assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations())
    with pytest.raises(hlb.HlbError):
        a.hlb_set_iolet_waveform(np.full((2, 3, 3), np.nan))
    with pytest.raises(ValueError):
        a.hlb_set_iolet_waveform(np.zeros((2, 2, 3)))
    a.close()
    b.close()
    cube = W.by_name("cube", small=True)                      # no iolets: nothing to drive
    c = hlb.hlb_geometry_create(cube.site_type, cube.periodic, cube.tau, cube.iolet_rho, flags)
    with pytest.raises(hlb.HlbError):
        c.hlb_set_iolet_waveform(np.zeros((2, 0, 3)))
    c.close()


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_normal_projected_pressure_iolets_match_oracle(hlb, scheme, lattice):
    """Constant-density iolets that only see the velocity along their normal (NEXT-3): the
    tree with its inlet normal +x and a seeded normal per outlet; random masks too."""
    import dataclasses
    wl = W.by_name("tree", small=True)
    rng = np.random.default_rng(8)
    normals = rng.standard_normal((wl.n_iolets, 3))
    normals[0] = (1.0, 0.0, 0.0)
    normals[3] = 0.0                                       # one outlet without a normal
    wl = dataclasses.replace(wl, iolet_normal=normals)
    for steps, order, links in ((wl.steps, "raster", "records"), (wl.steps + 1, "morton", "table")):
        rho_ref, u_ref = run_oracle(wl, steps, lattice=lattice)
        rho, u = run_gpu(hlb, wl, steps, scheme, "f64", order, links, lattice)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < 1e-12 and e_u < 1e-12, (steps, e_rho, e_u)
    plain = run_oracle(dataclasses.replace(wl, iolet_normal=None), wl.steps, lattice=lattice)
    assert np.max(np.abs(plain[1] - run_oracle(wl, wl.steps, lattice=lattice)[1])) > 1e-9
    rm = W.random_mask((14, 12, 10), p_fluid=0.65, n_iolets=3, p_iolet=0.07, tau=0.7, seed=92)
    rm = dataclasses.replace(rm, iolet_normal=rng.standard_normal((3, 3)))
    e_rho, e_u = errors(*run_gpu(hlb, rm, 11, scheme, "f64", "raster", "auto", lattice),
                        *run_oracle(rm, 11, lattice=lattice))
    assert e_rho < 1e-13 and e_u < 1e-12


# ------------------------------------------------------------- BFL interpolated walls (NEXT-2)
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("name", ["pipe", "aneurysm"])
def test_bfl_walls_match_oracle(hlb, name, lattice, scheme):
    """The paper's wall option: sub-voxel wall distances from the
    analytic surfaces of the pipe and the aneurysm, with a Ladd velocity inlet; both schemes,
    both storage types, records and table, even / odd / zero step counts."""
    wl = W.with_bfl_walls(W.with_velocity_inlet(W.by_name(name, small=True)))
    plain = W.with_velocity_inlet(W.by_name(name, small=True))
    for steps, store, order, links in ((wl.steps, "f64", "raster", "records"),
                                       (wl.steps + 1, "f64", "morton", "table"),
                                       (0, "f64", "raster", "auto"), (1, "f64", "raster", "auto"),
                                       (wl.steps, "f32", "raster", "auto")):
        rho_ref, u_ref = run_oracle(wl, steps, lattice=lattice)
        rho, u = run_gpu(hlb, wl, steps, scheme, store, order, links, lattice)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)
    # and the interpolation does change the flow (the test above is not vacuous)
    rho_p, u_p = run_oracle(plain, wl.steps, lattice=lattice)
    rho_b, u_b = run_oracle(wl, wl.steps, lattice=lattice)
    assert np.max(np.abs(u_p - u_b)) > 1e-6


@pytest.mark.parametrize("seed,periodic,shape", [(0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (33, 5, 4)),
                                                 (3, 0, (24, 20, 18)), (4, 5, (40, 9, 23))])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_bfl_random_masks_and_distances_match_oracle(hlb, seed, periodic, shape, scheme):
    wl = W.random_mask(shape, p_fluid=0.65, n_iolets=3, p_iolet=0.05, periodic=periodic,
                       tau=0.56 + 0.08 * seed, seed=500 + seed)
    rng = np.random.default_rng(seed)
    d27 = rng.uniform(0.01, 1.0, size=(wl.n_sites, 27))
    d27[rng.random(d27.shape) < 0.25] = 0.0
    perm = _match_directions(hlb)
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, "f64", "raster" if seed % 2 else "morton"))
    for x in (o, ):
        x.set_state(wl.rho0, wl.u0)
        x.set_wall_distance(d27)
    g.hlb_set_state(wl.rho0, wl.u0)
    g.hlb_set_wall_distance(d27)
    for n in (0, 1, 1, 7, 12, 1):                        # read-outs at even and odd step counts
        o.step(n)
        g.hlb_step(n)
        assert np.max(np.abs(g.hlb_get_populations()[:, perm] - o.get_populations())) < 1e-14
    g.hlb_set_state(wl.rho0, wl.u0)                      # distances survive a re-initialisation
    o.set_state(wl.rho0, wl.u0)
    if seed % 2:                                         # setting them again reuses the tables
        before = g.hlb_device_bytes()
        g.hlb_set_wall_distance(d27)
        assert g.hlb_device_bytes() == before
    o.step(5)
    g.hlb_step(5)
    e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o.get_macroscopic())
    assert e_rho < 1e-13 and e_u < 1e-12
    g.close()


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_bfl_at_half_a_link_is_bounce_back_bitwise_and_argument_errors(hlb, scheme):
    wl = W.by_name("tree", small=True)
    a = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, flags_of(hlb, scheme, "f64", "raster"))
    b = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, flags_of(hlb, scheme, "f64", "raster"))
    b.hlb_set_wall_distance(np.full((wl.n_sites, 27), 0.5))
    assert b.hlb_num_bfl_sites() > 100 and a.hlb_num_bfl_sites() == 0
    for n in (40, 1):
        a.hlb_step(n)
        b.hlb_step(n)
        (ra, ua), (rb, ub) = a.hlb_get_macroscopic(), b.hlb_get_macroscopic()
        assert np.array_equal(ra, rb) and np.array_equal(ua, ub)
    with pytest.raises(hlb.HlbError) as e:
        b.hlb_set_wall_distance(None)                    # not after the first step
    assert e.value.code == hlb.HLB_EINVAL
    b.hlb_set_state(None, None)
    b.hlb_set_wall_distance(None)                        # allowed again at step 0
    assert b.hlb_num_bfl_sites() == 0
    a.close()
    b.close()


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_bfl_read_outs_between_steps(hlb, scheme):
    """include/hlb.h, hlb_set_wall_distance: a read-out between steps runs the d < 1/2 pre-pass
    on the state buffer. In fp64 storage that changes nothing (bitwise); in fp32 storage it
    rounds the interpolated values one step early -- a perturbation of the size of the storage
    rounding, which must stay inside the fp32 bar against the oracle."""
    wl = W.with_bfl_walls(W.by_name("aneurysm", small=True))
    steps = 40
    rho_ref, u_ref = run_oracle(wl, steps, threads=1)
    for store in ("f64", "f32"):
        plain = run_gpu(hlb, wl, steps, scheme, store, "auto")
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                    flags_of(hlb, scheme, store, "auto"))
        g.hlb_set_wall_distance(wl.wall_distance)
        for _ in range(steps // 4):
            g.hlb_step(3)
            g.hlb_get_macroscopic()          # odd and even step counts
            g.hlb_step(1)
            g.hlb_get_populations()
        monitored = g.hlb_get_macroscopic()
        g.close()
        if store == "f64":
            assert np.array_equal(plain[0], monitored[0]) and np.array_equal(plain[1], monitored[1])
        e_rho, e_u = errors(*monitored, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (store, e_rho, e_u)


def test_bfl_is_the_same_in_both_schemes(hlb):
    """Two-lattice and A-A apply the same interpolation to the same values: populations after
    even and odd step counts agree to rounding (the two schemes round alike, see the bitwise
    variant tests; with interpolated walls the order of operations is the same too)."""
    wl = W.with_bfl_walls(W.with_velocity_inlet(W.by_name("aneurysm", small=True)))
    gs = []
    for scheme in ("two_lattice", "aa"):
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags_of(hlb, scheme, "f64"))
        g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
        g.hlb_set_wall_distance(wl.wall_distance)
        gs.append(g)
    assert gs[0].hlb_num_bfl_sites() == gs[1].hlb_num_bfl_sites() > 0
    for n in (1, 1, 9, 20):
        fs = []
        for g in gs:
            g.hlb_step(n)
            fs.append(g.hlb_get_populations())
        assert np.max(np.abs(fs[0] - fs[1])) < 1e-14
    for g in gs:
        g.close()


# ------------------------------------------------------------- stress read-out (NEXT-3)
STRESS_TOL = {"f64": 1e-9, "f32": 1e-3}   # f_neq is ~1e-3 of h, so the
                                          # population-level 1e-15 / 1e-7 is amplified ~1e3 x


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_stress_matches_oracle(hlb, scheme, lattice):
    """Deviatoric stress tensor of the pre-collision state, every site and component, after
    even and odd step counts (A-A reads it through the table after odd counts)."""
    wl = W.with_velocity_inlet(W.by_name("aneurysm", small=True), u_in=0.01)
    for store in ("f64", "f32"):
        o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, lattice=lattice, threads=0)
        o.set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                    flags_of(hlb, scheme, store, "raster", "auto", lattice))
        g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
        for n in (60, 41):
            o.step(n)
            g.hlb_step(n)
            ref, got = o.get_stress(), g.hlb_get_stress()
            scale = np.max(np.abs(ref))
            assert scale > 1e-7
            assert np.max(np.abs(got - ref)) / scale < STRESS_TOL[store], (store, n)
            assert np.array_equal(g.hlb_get_stress_device().cpu().numpy(), got)
            # wall shear stress with seeded normals on a third of the sites
            rng = np.random.default_rng(n)
            normals = rng.standard_normal((wl.n_sites, 3))
            normals[rng.random(wl.n_sites) < 0.66] = 0.0
            w_ref, w_got = o.get_wall_shear_stress(normals), g.hlb_get_wall_shear_stress(normals)
            assert np.all(w_got[np.all(normals == 0.0, axis=1)] == 0.0)
            assert np.max(np.abs(w_got - w_ref)) / np.max(w_ref) < STRESS_TOL[store]
        g.close()


def test_stress_is_zero_at_rest_and_uniform_flow(hlb):
    st = np.ones((6, 5, 4), dtype=np.uint8)
    g = hlb.hlb_geometry_create(st, 7, 0.7, [])
    assert np.all(g.hlb_get_stress() == 0.0)
    n = g.n_sites
    g.hlb_set_state(np.full(n, 1.02), np.tile(np.array([0.03, -0.02, 0.01]), (n, 1)))
    g.hlb_step(5)
    assert np.max(np.abs(g.hlb_get_stress())) < 1e-17
    g.close()


# ------------------------------------------------------------- random masks, every BC at once
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("seed,periodic,shape", [
    (0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (33, 5, 4)), (3, 2, (4, 19, 5)),
    (4, 4, (5, 4, 17)), (5, 7, (1, 1, 3)), (6, 3, (2, 2, 2)), (7, 0, (24, 20, 18)),
    (8, 5, (40, 9, 23)),
])
def test_random_masks_match_oracle(hlb, scheme, seed, periodic, shape):
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=3, p_iolet=0.06, periodic=periodic,
                       tau=0.55 + 0.07 * seed, seed=200 + seed)
    links, order = ("records", "raster") if seed % 2 else ("table", "morton")
    for steps in (0, 1, 2, 9, 10):
        rho_ref, u_ref = run_oracle(wl, steps, threads=1)
        rho, u = run_gpu(hlb, wl, steps, scheme, "f64", order, links)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < 1e-13 and e_u < 1e-12, (steps, e_rho, e_u)


def _match_directions(hlb):
    c_o, _, _ = oracle.velocity_set()
    c_g, _, _ = hlb.hlb_velocity_set()
    return [int(np.flatnonzero((c_g == c).all(axis=1))[0]) for c in c_o]   # oracle q -> library q


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_populations_match_oracle(hlb, scheme):
    """Population-level parity (stronger than moments), including set/get of populations."""
    wl = W.random_mask((12, 11, 10), p_fluid=0.65, n_iolets=2, periodic=1, tau=0.7, seed=77)
    perm = _match_directions(hlb)
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho)
    o.set_state(wl.rho0, wl.u0)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, "f64"))
    g.hlb_set_state(wl.rho0, wl.u0)
    assert np.array_equal(g.hlb_get_site_voxels(), o.site_voxels())
    for steps in (0, 1, 4, 3):
        o.step(steps)
        g.hlb_step(steps)
        fo, fg = o.get_populations(), g.hlb_get_populations()
        assert np.max(np.abs(fg[:, perm] - fo)) < 1e-15
    # round trip: the oracle's populations pushed into the library, then stepped
    fo = o.get_populations()
    fg = np.empty_like(fo)
    fg[:, perm] = fo
    g.hlb_set_populations(fg)
    assert g.hlb_steps_done() == 0
    assert np.max(np.abs(g.hlb_get_populations() - fg)) < 1e-16
    o.step(5)
    g.hlb_step(5)
    assert np.max(np.abs(g.hlb_get_populations()[:, perm] - o.get_populations())) < 1e-15
    g.close()


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_graph_replay_equals_direct_launches(hlb, scheme):
    """hlb_step replays captured graphs of 32 steps; same kernels, so bitwise the same as
    HLB_NO_GRAPH, whatever the split of the steps into calls (odd starts included)."""
    wl = W.by_name("aneurysm", small=True)
    f = flags_of(hlb, scheme, "f64", "raster")
    a = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f)
    b = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f | hlb.HLB_NO_GRAPH | hlb.HLB_NO_PDL)
    for n in (1, 70, 33, 32, 100):
        a.hlb_step(n)
        b.hlb_step(n)
        assert a.hlb_steps_done() == b.hlb_steps_done()
        assert a.hlb_launch_count() == b.hlb_launch_count() == a.hlb_steps_done()
        ra, ua = a.hlb_get_macroscopic()
        rb, ub = b.hlb_get_macroscopic()
        assert np.array_equal(ra, rb) and np.array_equal(ua, ub)
    a.hlb_set_state(None, None)                      # reset, then straight into a graph
    b.hlb_set_state(None, None)
    a.hlb_step(64)
    b.hlb_step(64)
    assert np.array_equal(a.hlb_get_macroscopic()[1], b.hlb_get_macroscopic()[1])
    a.close()
    b.close()


# ------------------------------------------------------------- resident multi-step kernel
@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_resident_kernel_matches_oracle(hlb, scheme, store, lattice):
    """Small geometries run hlb_step(n >= 2) as one cooperative launch with grid barriers
    between the steps: BASELINE configs[0] at full size and step count, and the scaled-down
    other configs, against the oracle (even and odd step counts)."""
    for name, small in (("pipe", False), ("cube", True), ("aneurysm", True), ("tree", True)):
        wl = W.by_name(name, small=small)
        for steps in (wl.steps, 7):
            rho_ref, u_ref = (run_oracle(wl, steps, lattice=lattice) if not small
                              else oracle_cached(name, steps, lattice))
            g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                        flags_of(hlb, scheme, store, "raster", "auto", lattice, resident=True))
            if wl.rho0 is not None or wl.u0 is not None:
                g.hlb_set_state(wl.rho0, wl.u0)
            g.hlb_step(steps)
            assert g.hlb_steps_done() == steps and g.hlb_launch_count() == 1, (name, g.hlb_launch_count())
            e_rho, e_u = errors(*g.hlb_get_macroscopic(), rho_ref, u_ref)
            g.close()
            assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, lattice, steps, e_rho, e_u)


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_resident_kernel_equals_direct_launches(hlb, scheme, lattice):
    """Same per-site arithmetic: populations bitwise equal to the one-shot kernels launched
    step by step, for any split of the steps into calls (odd starts, single steps in between,
    which are launched directly), with every boundary kind on the sites (walls, density and
    velocity iolets, iolet normals), table and record links, 64-bit offsets."""
    wl = W.random_mask((21, 17, 19), p_fluid=0.7, n_iolets=3, p_iolet=0.06, periodic=4, tau=0.57, seed=33)
    kind = np.array([1, 0, 0], dtype=np.uint8)
    u = np.array([[0.004, -0.002, 0.001], [0, 0, 0], [0, 0, 0]], dtype=np.float64)
    normals = np.array([[0, 0, 0], [0.0, 1.0, 0.0], [0, 0, 0]], dtype=np.float64)
    for links, extra, full in (("records", 0, False), ("table", 0, True), ("auto", hlb.HLB_INDEX64, True)):
        f = flags_of(hlb, scheme, "f64", "raster", links, lattice, resident=True) | extra
        a = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, f)
        b = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, f | hlb.HLB_NO_GRAPH)
        for x in (a, b):
            x.hlb_set_state(wl.rho0, wl.u0)
            if full:
                x.hlb_set_iolet_velocity(kind, u)
                x.hlb_set_iolet_normal(normals)
        done = 0
        for n in (3, 1, 64, 2, 33):
            a.hlb_step(n)
            b.hlb_step(n)
            done += n
            assert a.hlb_steps_done() == b.hlb_steps_done() == done
            assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations()), (links, n)
        # (the resident kernels exist for 32-bit offsets only: HLB_INDEX64 steps one by one)
        assert a.hlb_launch_count() == (done if extra & hlb.HLB_INDEX64 else 5) and b.hlb_launch_count() == done
        a.close()
        b.close()


def test_resident_kernel_is_not_used_where_it_does_not_apply(hlb):
    """Interpolated walls and waveforms keep the one-shot kernels; so does a geometry too large
    to be resident (one launch per step), and the results stay those of the direct launches."""
    wl = W.with_bfl_walls(W.with_velocity_inlet(W.by_name("pipe", small=True)))
    f = flags_of(hlb, "aa", "f64", "raster", resident=True)
    g = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f)
    g.hlb_set_wall_distance(wl.wall_distance)
    g.hlb_step(6)
    assert g.hlb_launch_count() >= 6
    g.close()
    big = W.by_name("aneurysm")                              # 739 k sites: not resident
    a = hlb.hlb_geometry_create(big.site_type, 0, big.tau, big.iolet_rho, f)
    b = hlb.hlb_geometry_create(big.site_type, 0, big.tau, big.iolet_rho, f | hlb.HLB_NO_GRAPH)
    a.hlb_step(40)
    b.hlb_step(40)
    assert a.hlb_launch_count() == b.hlb_launch_count() == 40
    assert np.array_equal(a.hlb_get_macroscopic()[1], b.hlb_get_macroscopic()[1])
    a.close()
    b.close()


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_graph_replay_with_boundary_options(hlb, scheme):
    """Graph replay with interpolated walls (read-outs in between: the step after a read-out
    and the first step are launched directly) equals direct launches bitwise; and a graph
    captured with the lean iolet kernels is dropped when an iolet becomes a velocity iolet."""
    wl = W.with_bfl_walls(W.with_velocity_inlet(W.by_name("aneurysm", small=True)))
    f = flags_of(hlb, scheme, "f64", "raster")
    a = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f)
    b = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f | hlb.HLB_NO_GRAPH)
    o = oracle.Oracle(wl.site_type, 0, wl.tau, wl.iolet_rho)
    for x in (a, b):
        x.hlb_set_wall_distance(wl.wall_distance)
    o.set_wall_distance(wl.wall_distance)
    total = 0
    for n in (70, 33, 1, 64):                            # pressure iolets: lean kernels
        a.hlb_step(n)
        b.hlb_step(n)
        total += n
        assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations())
    for x in (a, b):
        x.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)   # now the full kernels
    o.step(total)
    o.set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
    for n in (66, 35):
        a.hlb_step(n)
        b.hlb_step(n)
        o.step(n)
        assert np.array_equal(a.hlb_get_populations(), b.hlb_get_populations())
        e_rho, e_u = errors(*a.hlb_get_macroscopic(), *o.get_macroscopic())
        assert e_rho < 1e-13 and e_u < 1e-12, (n, e_rho, e_u)
    a.close()
    b.close()


@pytest.mark.parametrize("links", ["table", "records"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_64_bit_offset_kernels_equal_32_bit(hlb, scheme, links):
    """Above 2^32 / 15 sites the kernels index with 64-bit offsets; HLB_INDEX64 forces that
    instantiation on a small geometry: bitwise the same as the 32-bit one."""
    wl = W.by_name("bigtree", small=True)
    for store in ("f64", "f32"):      # (f32 + A-A + records: the shared-memory record path of k_aa_odd)
        f = flags_of(hlb, scheme, store, "raster", links)
        out = []
        for extra in (0, hlb.HLB_INDEX64):
            g = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f | extra)
            g.hlb_step(23)
            out.append(g.hlb_get_macroscopic())
            g.close()
        assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1]), store


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_l2_prefetch_changes_nothing(hlb, scheme, monkeypatch):
    """The L2 prefetches are hints: bitwise the same results with a distance that really
    fires on a small geometry (HLB_PREFETCH_SITES) and with HLB_NO_PREFETCH."""
    wl = W.by_name("tree", small=True)
    f = flags_of(hlb, scheme, "f64", "raster", "records")
    monkeypatch.setenv("HLB_PREFETCH_SITES", "1024")
    a = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f)
    monkeypatch.delenv("HLB_PREFETCH_SITES")
    b = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, f | hlb.HLB_NO_PREFETCH)
    a.hlb_step(37)
    b.hlb_step(37)
    (ra, ua), (rb, ub) = a.hlb_get_macroscopic(), b.hlb_get_macroscopic()
    assert np.array_equal(ra, rb) and np.array_equal(ua, ub)
    a.close()
    b.close()


# ------------------------------------------------------------- invariants on the GPU itself
@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_rest_state_is_bitwise_invariant(hlb, scheme, store):
    wl = W.by_name("tree", small=True)
    g = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, np.ones(wl.n_iolets),
                                flags_of(hlb, scheme, store))
    g.hlb_step(51)
    rho, u = g.hlb_get_macroscopic()
    assert np.all(rho == 1.0) and np.all(u == 0.0)
    g.close()


def test_state_round_trip_and_iolet_update(hlb):
    wl = W.by_name("pipe", small=True)
    n = wl.n_sites
    rng = np.random.default_rng(3)
    rho0 = 1.0 + 0.01 * rng.standard_normal(n)
    u0 = 0.01 * rng.standard_normal((n, 3))
    for scheme in ("two_lattice", "aa"):
        g = hlb.hlb_geometry_create(wl.site_type, 0, wl.tau, wl.iolet_rho, flags_of(hlb, scheme, "f64"))
        g.hlb_set_state(rho0, u0)
        rho, u = g.hlb_get_macroscopic()
        assert np.max(np.abs(rho - rho0)) < 1e-15 and np.max(np.abs(u - u0)) < 1e-16
        rd, ud = g.hlb_get_macroscopic_device()
        assert np.array_equal(rd.cpu().numpy(), rho) and np.array_equal(ud.cpu().numpy(), u)
        # new iolet densities take effect: compare with an oracle built with them
        g.hlb_set_state(None, None)
        g.hlb_set_iolet_density([1.002, 0.997])
        g.hlb_step(20)
        o = oracle.Oracle(wl.site_type, 0, wl.tau, [1.002, 0.997])
        o.step(20)
        e_rho, e_u = errors(*g.hlb_get_macroscopic(), *o.get_macroscopic())
        assert e_rho < 1e-12 and e_u < 1e-12
        g.close()


def test_asynchronous_read_out_on_a_copy_stream(hlb):
    """hlb_get_macroscopic_async + hlb_wait_copies (include/hlb.h): the same numbers as the
    synchronous read-out, also when the next upload and steps are enqueued before the copies
    are waited for; without a copy stream the call is refused."""
    import torch
    wl = W.by_name("tree", small=True)
    n = wl.n_sites
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, "aa", "f64", "auto"), copy_stream=torch.cuda.Stream())
    outs = [(torch.empty(n, dtype=torch.float64).pin_memory().numpy(),
             torch.empty((n, 3), dtype=torch.float64).pin_memory().numpy()) for _ in range(2)]
    want = []
    for k, steps in enumerate((7, 12)):
        g.hlb_set_state(None, None)
        g.hlb_step(steps)
        g.hlb_get_macroscopic_async(*outs[k])      # not waited for: the next round is enqueued behind it
        want.append(run_gpu(hlb, wl, steps, "aa", "f64", "auto"))
    g.hlb_wait_copies()
    for k in range(2):
        assert np.array_equal(outs[k][0], want[k][0]) and np.array_equal(outs[k][1], want[k][1])
    g.close()
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags_of(hlb, "aa", "f64", "auto"))
    with pytest.raises(hlb.HlbError) as e:
        g.hlb_get_macroscopic_async(*outs[0])
    assert e.value.code == hlb.HLB_EINVAL
    g.close()


def test_staged_upload_on_a_copy_stream(hlb):
    """hlb_stage_state + hlb_set_state_staged (include/hlb.h): the same run as hlb_set_state, also
    when the upload of the next state is enqueued while the steps of the current one are in
    flight; refused without a copy stream or without a staged state."""
    import torch
    wl = W.by_name("cube", small=True)
    n = wl.n_sites
    rng = np.random.default_rng(3)
    states = [(1.0 + 0.01 * rng.random(n), 0.02 * (rng.random((n, 3)) - 0.5)) for _ in range(3)]
    pinned = [(torch.from_numpy(r).pin_memory().numpy(), torch.from_numpy(u).pin_memory().numpy()) for r, u in states]
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, "aa", "f64", "auto"), copy_stream=torch.cuda.Stream())
    with pytest.raises(hlb.HlbError):
        g.hlb_set_state_staged()                       # nothing staged
    got = []
    g.hlb_stage_state(*pinned[0])
    for k in range(3):
        g.hlb_set_state_staged()
        g.hlb_step(9 + k)
        if k + 1 < 3:
            g.hlb_stage_state(*pinned[k + 1])          # uploads under the steps just enqueued
        got.append(g.hlb_get_macroscopic())
    g.hlb_wait_copies()
    g.close()
    for k in range(3):
        wl_k = W.Workload("cube", wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, 0, rho0=states[k][0], u0=states[k][1])
        want = run_gpu(hlb, wl_k, 9 + k, "aa", "f64", "auto")
        assert np.array_equal(got[k][0], want[0]) and np.array_equal(got[k][1], want[1])
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags_of(hlb, "aa", "f64", "auto"))
    with pytest.raises(hlb.HlbError) as e:
        g.hlb_stage_state(*pinned[0])
    assert e.value.code == hlb.HLB_EINVAL
    g.close()


def test_degenerate_geometries(hlb):
    st = np.zeros((3, 3, 3), dtype=np.uint8)
    st[1, 1, 1] = 1                                   # one site, every link bounces back
    for scheme in ("two_lattice", "aa"):
        g = hlb.hlb_geometry_create(st, 0, 0.8, [], flags_of(hlb, scheme, "f64"))
        g.hlb_set_state(np.array([1.01]), np.array([[0.01, -0.02, 0.005]]))
        g.hlb_step(0)
        g.hlb_step(7)
        o = oracle.Oracle(st, 0, 0.8, [])
        o.set_state(np.array([1.01]), np.array([[0.01, -0.02, 0.005]]))
        o.step(7)
        (r, u), (ro, uo) = g.hlb_get_macroscopic(), o.get_macroscopic()
        assert abs(r[0] - ro[0]) < 1e-15 and np.max(np.abs(u - uo)) < 1e-15
        g.close()
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_geometry_create(np.zeros((2, 2, 2), dtype=np.uint8), 0, 0.8, [])
    assert e.value.code == hlb.HLB_ENOFLUID
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_geometry_create(st, 0, 0.5, [])
    assert e.value.code == hlb.HLB_EINVAL
    g = hlb.hlb_geometry_create(st, 0, 0.8, [])
    with pytest.raises(hlb.HlbError):
        g.hlb_step(-1)
    g.close()


# ------------------------------------------------------------- full-size configs
def test_config0_pipe_full(hlb):
    """BASELINE configs[0] exactly: 12,608 sites, tau 0.8, 200 steps."""
    wl = W.pipe()
    assert wl.n_sites == 12608
    rho_ref, u_ref = run_oracle(wl, wl.steps)
    for scheme in ("two_lattice", "aa"):
        e_rho, e_u = errors(*run_gpu(hlb, wl, wl.steps, scheme, "f64"), rho_ref, u_ref)
        assert e_rho < 1e-12 and e_u < 1e-12, (scheme, e_rho, e_u)


def test_config1_cube_full_size(hlb):
    """BASELINE configs[1] at full size (128^3, tau 0.6, Taylor-Green): parity with the
    oracle after 60 steps (every site), then the full 1000 steps checked through properties
    that hold at any size: exact mass conservation and the closed-form decay."""
    wl = W.periodic_cube()
    n = wl.n_sites
    assert n == 128 ** 3
    rho_ref, u_ref = run_oracle(wl, 60)
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, [], flags_of(hlb, "two_lattice", "f64"))
    g.hlb_set_state(wl.rho0, wl.u0)
    g.hlb_step(60)
    e_rho, e_u = errors(*g.hlb_get_macroscopic(), rho_ref, u_ref)
    assert e_rho < 1e-12 and e_u < 1e-12, (e_rho, e_u)
    ke = {}
    for t in (200, 600, 1000):
        g.hlb_step(t - g.hlb_steps_done())
        rho, u = g.hlb_get_macroscopic()
        ke[t] = 0.5 * np.sum(rho[:, None] * u * u)
        assert abs(rho.sum() - n) / n < 1e-14           # mass: exactly conserved up to rounding
    nu, k = (wl.tau - 0.5) / 3.0, wl.info["k"]
    for a, b in ((200, 600), (600, 1000)):
        assert ke[b] / ke[a] == pytest.approx(np.exp(-4.0 * nu * k * k * (b - a)), rel=2e-3)
    g.close()


def test_config2_aneurysm_full_size(hlb):
    """BASELINE configs[2] at full size (739,223 sites): all sites against the oracle after
    150 steps; the 2000-step run is the slow record test below."""
    wl = W.aneurysm()
    assert wl.n_sites == 739223
    rho_ref, u_ref = run_oracle(wl, 150)
    for scheme in ("two_lattice", "aa"):
        e_rho, e_u = errors(*run_gpu(hlb, wl, 150, scheme, "f64"), rho_ref, u_ref)
        assert e_rho < 1e-12 and e_u < 1e-12, (scheme, e_rho, e_u)


def _smooth_state(x, y, z):
    """A smooth, non-trivial initial field as a function of ABSOLUTE voxel coordinates, so
    that a crop and the full geometry start from the same state."""
    x, y, z = (np.asarray(a, dtype=np.float64) for a in (x, y, z))
    rho = 1.0 + 0.01 * np.sin(0.07 * x + 0.05 * y) * np.cos(0.06 * z)
    u = 0.02 * np.stack([np.sin(0.05 * y + 0.03 * z), np.cos(0.04 * x - 0.06 * z),
                         np.sin(0.03 * x + 0.07 * y)], axis=1)
    return rho, u


def _crop_check(hlb, wl, rho, u, steps, centre, half, tol, lattice="d3q15"):
    """Exact check of a full-size run on a sample: a site update is local (information moves
    one voxel per step), so the oracle run on the sub-box [centre - half, centre + half] of
    the same voxel array (outside the crop = solid) reproduces, after `steps` steps, every
    site that is more than `steps` voxels away from the crop faces lying inside the box."""
    st = wl.site_type
    nz, ny, nx = st.shape
    lo = [max(0, c - half) for c in centre]
    hi = [min(n, c + half + 1) for c, n in zip(centre, (nx, ny, nz))]
    sub = np.ascontiguousarray(st[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]])
    o = oracle.Oracle(sub, 0, wl.tau, wl.iolet_rho, threads=0, lattice=lattice)
    v = o.site_voxels()
    sx, sy, sz = hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]
    x, y, z = v % sx + lo[0], (v // sx) % sy + lo[1], v // (sx * sy) + lo[2]
    o.set_state(*_smooth_state(x, y, z))
    o.step(steps)
    rho_c, u_c = o.get_macroscopic()
    o.close()
    keep = np.ones(v.shape, dtype=bool)
    for c, l, h, n in ((x, lo[0], hi[0], nx), (y, lo[1], hi[1], ny), (z, lo[2], hi[2], nz)):
        if l > 0:
            keep &= c - l > steps
        if h < n:
            keep &= (h - 1) - c > steps
    assert keep.sum() > 1000, "sample too small to mean anything"
    full_voxel = (z * ny + y) * nx + x
    canon = np.searchsorted(wl.fluid_voxels(), full_voxel[keep])
    e_rho = np.max(np.abs(rho[canon] - rho_c[keep])) / np.max(np.abs(rho_c[keep]))
    un = np.max(np.linalg.norm(u_c[keep], axis=1))
    e_u = np.max(np.abs(u[canon] - u_c[keep])) / (un if un > 0 else 1.0)
    assert e_rho < tol and e_u < tol, (centre, e_rho, e_u)
    return int(keep.sum()), un


def _sample_centres(wl, n):
    """The inlet end, the outlet-most end and evenly spaced fluid voxels in between."""
    v = wl.fluid_voxels()
    nz, ny, nx = wl.site_type.shape
    picks = v[np.linspace(0, len(v) - 1, n).astype(np.int64)]
    x = picks % nx
    return [(int(a), int(b), int(c)) for a, b, c in zip(x, (picks // nx) % ny, picks // (nx * ny))]


@pytest.mark.parametrize("name,scheme,store,lattice", [
    ("tree", "two_lattice", "f64", "d3q15"), ("tree", "two_lattice", "f32", "d3q15"),
    ("bigtree", "aa", "f64", "d3q15"), ("tree", "aa", "f64", "d3q19"),
])
def test_configs_3_4_full_size_sampled_against_oracle(hlb, name, scheme, store, lattice):
    """BASELINE configs[3] / [4] at full size in the launch configuration bench.py times
    (default order, link records, L2 prefetch): 25 steps (odd: A-A read-out through the
    table), then sub-boxes compared site by site with the oracle (see _crop_check)."""
    wl = W.by_name(name)
    steps, half = 25, 56
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, scheme, store, "auto", "auto", lattice))
    assert g.hlb_uses_records()
    nz, ny, nx = wl.site_type.shape
    v = wl.fluid_voxels()
    g.hlb_set_state(*_smooth_state(v % nx, (v // nx) % ny, v // (nx * ny)))
    g.hlb_step(steps)
    rho, u = g.hlb_get_macroscopic()
    g.close()
    assert np.all(np.isfinite(rho)) and np.all(np.isfinite(u))
    checked = 0
    for centre in _sample_centres(wl, 5):
        n, un = _crop_check(hlb, wl, rho, u, steps, centre, half, TOL[store], lattice)
        assert un > 1e-3                                  # the sample is not at rest
        checked += n
    assert checked > 20000


def test_scheme_auto_picks_and_matches_the_explicit_scheme(hlb):
    """HLB_SCHEME_AUTO: two-lattice where the resident multi-step kernel applies (small
    geometries), A-A in place otherwise; either way bitwise the explicitly chosen scheme."""
    wl = W.by_name("aneurysm", small=True)
    for extra, want_aa in ((0, False), (hlb.HLB_NO_RESIDENT, True)):
        g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                    hlb.HLB_SCHEME_AUTO | extra)
        assert g.hlb_uses_aa() == want_aa
        g.hlb_step(31)
        got = g.hlb_get_macroscopic()
        g.close()
        ref = run_gpu(hlb, wl, 31, "aa" if want_aa else "two_lattice", "f64", "auto")
        assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1])
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    for name, lattice in (("paper_sized", "d3q15"), ("paper_sized", "d3q19"), ("paper_sized_23", "d3q15"),
                          ("paper_sized_23", "d3q19")):
        big = W.by_name(name)
        g = hlb.hlb_geometry_create(big.site_type, big.periodic, big.tau, big.iolet_rho,
                                    hlb.HLB_SCHEME_AUTO | flags_of(hlb, "two_lattice", "f64", "auto", "auto", lattice, True))
        # beyond the resident kernel: two-lattice only if the grid is one wave of the two-lattice
        # kernel (blocks per SM: 6 for D3Q15 fp64, 5 for D3Q19; 5 % slack) and more than one of A-A (6 / 4)
        blocks = -(-big.n_sites // 128)
        per_sm_pull, per_sm_aa = (6, 6) if lattice == "d3q15" else (5, 4)
        want_aa = not (blocks > sms * per_sm_aa and blocks * 100 <= sms * per_sm_pull * 105)
        assert g.hlb_uses_aa() == want_aa, (name, lattice, blocks)
        g.close()


# ------------------------------------------------------------- north_star's acceptance runs
# "GPU results must match the oracle on the same seeded inputs ... after the configured steps
# ... on all five configs" (BASELINE.json north_star): full size
# AND full step count, site by site, in the scheme the config names. Part of the default
# -m gpu run (config 0 is test_config0_pipe_full above); the E_rho / E_u of every run are
# printed in the terminal summary (tests/conftest.py).
@pytest.mark.slow
@pytest.mark.parametrize("name", ["pipe", "cube", "aneurysm", "tree", "bigtree"])
def test_full_configs_full_steps_record(hlb, name, record):
    wl = W.by_name(name)
    rho_ref, u_ref = run_oracle(wl, wl.steps)
    stores = ("f64", "f32") if name == "tree" else ("f64",)
    for store in stores:
        e_rho, e_u = errors(*run_gpu(hlb, wl, wl.steps, wl.scheme, store, "auto"), rho_ref, u_ref)
        record(f"RECORD {name} N={wl.n_sites} steps={wl.steps} {wl.scheme}/{store} "
               f"E_rho={e_rho:.3e} E_u={e_u:.3e} (bar {TOL[store]:.0e})")
        assert e_rho < TOL[store] and e_u < TOL[store]
    if name == "tree":   # the scheme HLB_SCHEME_AUTO picks at this size, with 4-byte storage
        e_rho, e_u = errors(*run_gpu(hlb, wl, wl.steps, "aa", "f32", "auto"), rho_ref, u_ref)
        record(f"RECORD {name} N={wl.n_sites} steps={wl.steps} aa/f32 E_rho={e_rho:.3e} E_u={e_u:.3e} (bar 1e-05)")
        assert e_rho < TOL["f32"] and e_u < TOL["f32"]
    if name == "aneurysm":   # the lattice the paper ran, in place
        rho19, u19 = run_oracle(wl, wl.steps, lattice="d3q19")
        e_rho, e_u = errors(*run_gpu(hlb, wl, wl.steps, "aa", "f64", "auto", "auto", "d3q19"), rho19, u19)
        record(f"RECORD {name} N={wl.n_sites} steps={wl.steps} D3Q19 aa/f64 E_rho={e_rho:.3e} E_u={e_u:.3e} (bar 1e-12)")
        assert e_rho < TOL["f64"] and e_u < TOL["f64"]


@pytest.mark.slow
def test_config3_full_size_with_every_wall_link_interpolated_record(hlb, record):
    """NEXT-2 at the size bench.py times it (--workload tree --inlet velocity --walls bfl_random):
    all 4.9 M sites of configs[3], a Ladd velocity inlet and a seeded random wall distance on
    every wall link (0.8 M sites carry one; row ranks far beyond 16 bits), every site against
    the oracle, both schemes, both storage types; odd step count for the in-place scheme."""
    wl = W.with_velocity_inlet(W.by_name("tree"))
    d27 = np.random.default_rng(1906).uniform(0.05, 1.0, size=(wl.n_sites, 27))
    wl = dataclasses.replace(wl, wall_distance=d27)
    refs = {steps: run_oracle(wl, steps) for steps in (100, 101)}
    for scheme, store, steps in (("two_lattice", "f64", 100), ("aa", "f64", 101), ("aa", "f32", 101),
                                 ("two_lattice", "f32", 100)):
        e_rho, e_u = errors(*run_gpu(hlb, wl, steps, scheme, store, "auto"), *refs[steps])
        record(f"RECORD tree + velocity inlet + BFL on every wall link N={wl.n_sites} steps={steps} "
               f"{scheme}/{store} E_rho={e_rho:.3e} E_u={e_u:.3e} (bar {TOL[store]:.0e})")
        assert e_rho < TOL[store] and e_u < TOL[store]


# ------------------------------------------------------------- the sizes the library claims
def _needs(host_gb, device_gb):
    """These two cases need a large box (the B200 boxes of this pool have 196 GB of host memory
    and 180 GB of HBM); elsewhere they skip rather than drive a small machine out of memory."""
    import psutil
    import torch
    if psutil.virtual_memory().available < host_gb * 2 ** 30:
        pytest.skip(f"needs {host_gb} GB of free host memory")
    if torch.cuda.mem_get_info()[0] < device_gb * 2 ** 30:
        pytest.skip(f"needs {device_gb} GB of free device memory")


@pytest.mark.slow
def test_cube672_runs_the_64_bit_offset_kernels_for_real(hlb, record):
    """303.5 M sites: Q * N = 4.55e9 > 2^32, so the `long long` offset instantiations are the ones
    launched (without HLB_INDEX64), the int32 table holds entries up to 3.0e8, the link-record
    deltas wrap, and 17 GB of table + 36 GB of populations are uploaded. Checked by exact mass
    conservation (periodic box) and by the oracle on interior sub-boxes of the same field,
    chosen so that the compared sites sit in the first, a middle and the last plane rows."""
    _needs(70, 80)
    wl = W.by_name("cube672")
    n = wl.info["n"]
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, "aa", "f64", "auto", "auto"))
    assert g.hlb_offset_bits() == 64 and g.hlb_uses_records() and g.n_sites == n ** 3
    ax = np.arange(n, dtype=np.float64)
    rho = (1.0 + 0.01 * np.sin(0.07 * ax[None, None, :] + 0.05 * ax[None, :, None])
           * np.cos(0.06 * ax[:, None, None])).reshape(-1)
    u = np.empty((n ** 3, 3), dtype=np.float64)
    z, y, x = ax[:, None, None], ax[None, :, None], ax[None, None, :]
    u[:, 0] = (0.02 * np.sin(0.05 * y + 0.03 * z) + 0.0 * x).reshape(-1)
    u[:, 1] = (0.02 * np.cos(0.04 * x - 0.06 * z) + 0.0 * y).reshape(-1)
    u[:, 2] = (0.02 * np.sin(0.03 * x + 0.07 * y) + 0.0 * z).reshape(-1)
    g.hlb_set_state(rho, u)
    mass0 = float(np.sum(rho, dtype=np.float64))
    del rho, u
    steps = 25
    g.hlb_step(steps)
    rho, u = g.hlb_get_macroscopic()
    dev_gb = g.hlb_device_bytes() / 2 ** 30
    g.close()
    assert np.all(np.isfinite(rho)) and np.all(np.isfinite(u))
    drift = abs(float(np.sum(rho, dtype=np.float64)) - mass0) / n ** 3
    assert drift < 1e-14, drift                     # shifted populations: mass is conserved to roundoff
    checked = 0
    for centre in ((60, 60, 60), (336, 300, 340), (600, 610, 611)):
        k, un = _crop_check(hlb, wl, rho, u, steps, centre, 56, TOL["f64"])
        assert un > 1e-3
        checked += k
    record(f"HUGE cube672 N={n ** 3} steps={steps} aa/f64 offsets=64-bit device={dev_gb:.1f} GiB "
           f"mass drift/site={drift:.1e} sites compared with the oracle={checked}")


@pytest.mark.slow
def test_bigtree_at_baselines_nominal_size(hlb, record):
    """configs[4]'s generator at BASELINE's nominal 80-100 M sites (workloads 'bigtree_x':
    85.5 M), A-A fp64 in the bench's launch configuration, 25 steps from a smooth field, sampled
    sub-boxes against the oracle."""
    _needs(40, 30)
    wl = W.by_name("bigtree_x")
    steps = 25
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                flags_of(hlb, "aa", "f64", "auto", "auto"))
    assert g.hlb_uses_records() and g.hlb_offset_bits() == 32
    nz, ny, nx = wl.site_type.shape
    v = wl.fluid_voxels()
    g.hlb_set_state(*_smooth_state(v % nx, (v // nx) % ny, v // (nx * ny)))
    g.hlb_step(steps)
    rho, u = g.hlb_get_macroscopic()
    g.close()
    assert np.all(np.isfinite(rho)) and np.all(np.isfinite(u))
    checked = 0
    for centre in _sample_centres(wl, 5):
        k, un = _crop_check(hlb, wl, rho, u, steps, centre, 56, TOL["f64"])
        assert un > 1e-3
        checked += k
    assert checked > 20000
    record(f"HUGE bigtree_x N={wl.n_sites} steps={steps} aa/f64 sites compared with the oracle={checked}")


# ------------------------------------------------------------- long horizon, every variant
@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
@pytest.mark.parametrize("name,lattice", [("aneurysm", "d3q15"), ("tree", "d3q15"), ("cube", "d3q15"),
                                          ("aneurysm", "d3q19")])
def test_long_horizon_drift_against_oracle(hlb, name, lattice, scheme, store, record):
    """>= 1000 steps on the scaled-down configs for every {scheme x storage}: the fp32-storage
    rounding (budget 1e-5, reading A15) and the fp64 evaluation-order differences must not
    grow past the bar over a horizon longer than any config's; 1001 steps reads the A-A state
    out at odd parity."""
    wl = W.by_name(name, small=True)
    for steps in (1000, 1001):
        rho_ref, u_ref = oracle_cached(name, steps, lattice)
        rho, u = run_gpu(hlb, wl, steps, scheme, store, "auto", "auto", lattice)
        e_rho, e_u = errors(rho, u, rho_ref, u_ref)
        assert e_rho < TOL[store] and e_u < TOL[store], (name, scheme, store, steps, e_rho, e_u)
    record(f"LONG {name}(small) N={wl.n_sites} steps=1001 {lattice} {scheme}/{store} "
           f"E_rho={e_rho:.3e} E_u={e_u:.3e} (bar {TOL[store]:.0e})")
