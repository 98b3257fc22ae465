"""The no-allocation entry point hlb_get_wall_shear_stress_noalloc (include/hlb.h) against the
existing path hlb_get_wall_shear_stress: same kernels, the stress tensor staged in the library's
static __device__ array instead of an allocated buffer.

This file is named to be collected LAST (the suite runs with pytest -x): it must pass alone in
a fresh process and after every other test of the suite.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-12          # of max|wss|; the bar of the fp64 tests (the two paths run the same kernels)


@pytest.fixture(scope="module")
def hlb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1906_11925_b200 as m
    return m


def _normals(wl, seed):
    """Seeded synthetic wall normals: random directions, zero (= not a wall site) at a third."""
    rng = np.random.default_rng(seed)
    n = rng.normal(size=(wl.n_sites, 3))
    n[rng.random(wl.n_sites) < 0.33] = 0.0
    return n


def test_no_alloc_wall_shear_stress_equals_the_allocating_path_twice_in_a_row(hlb):
    import torch
    wl = W.by_name("aneurysm", small=True)
    assert wl.n_sites <= hlb.hlb_noalloc_max_sites() == 262144
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                hlb.HLB_AA | hlb.HLB_NO_RESIDENT)
    dev = g.device
    wss_dev = torch.empty(wl.n_sites, dtype=torch.float64, device=dev)
    # a second geometry (other lattice, two-lattice scheme) shares the same static array
    g2 = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho,
                                 hlb.HLB_LATTICE_D3Q19 | hlb.HLB_NO_RESIDENT)
    for call, (geom, steps) in enumerate(((g, 21), (g, 6), (g2, 15), (g, 0))):
        geom.hlb_step(steps)
        nrm = _normals(wl, 10 + call)
        want = geom.hlb_get_wall_shear_stress(nrm)                 # existing path (host arrays)
        nrm_dev = torch.from_numpy(nrm).to(dev)
        wss_dev.fill_(float("nan"))                                # every entry must be written
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated(dev), geom.hlb_device_bytes()
        geom.hlb_get_wall_shear_stress_noalloc(nrm_dev, wss_dev)
        after = torch.cuda.memory_allocated(dev), geom.hlb_device_bytes()
        assert before == after                                     # the allocator callback was not used
        got = wss_dev.cpu().numpy()
        scale = float(np.max(np.abs(want)))
        assert scale > 0.0 and np.all(np.isfinite(got))
        assert np.max(np.abs(got - want)) <= TOL * scale, (call, np.max(np.abs(got - want)), scale)
        assert np.all(got[np.all(nrm == 0.0, axis=1)] == 0.0)
    g.close()
    g2.close()


def test_no_alloc_entry_point_rejects_what_does_not_fit(hlb):
    import torch
    wl = W.periodic_cube(n=65, with_state=False)                   # 274,625 sites > 262,144
    assert wl.n_sites > hlb.hlb_noalloc_max_sites()
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, hlb.HLB_AA)
    nrm = torch.zeros((wl.n_sites, 3), dtype=torch.float64, device=g.device)
    out = torch.full((wl.n_sites,), 7.0, dtype=torch.float64, device=g.device)
    with pytest.raises(hlb.HlbError) as e:
        g.hlb_get_wall_shear_stress_noalloc(nrm, out)
    assert e.value.code == hlb.HLB_ETOOLARGE and "HLB_NOALLOC_MAX_SITES" in str(e.value)
    assert bool(torch.all(out == 7.0))                             # nothing was launched
    with pytest.raises(ValueError):
        g.hlb_get_wall_shear_stress_noalloc(nrm[:-1], out)
    g.close()
