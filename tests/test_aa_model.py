"""CPU model of the in-place A-A scheme (no GPU): the property the kernels k_aa_even / k_aa_odd
rest on, re-proved on the library's own pull table (SURVEY.md §8(a) row S7, §5 "Race detection",
§9 item 4: "re-prove the read-set = write-set property on a CPU model").

Two statements, on random masks with walls, iolet ghost voxels and periodic wrap, both lattices
and every site order of the preprocessor:

1. Address sets. In each phase the slots a site reads are exactly the slots it writes, the
   sets of different sites are disjoint and together they cover all Q x N slots -- so one array
   suffices and no two threads ever touch the same slot in a launch (the racecheck substitute:
   compute-sanitizer is closed on this GPU pool).
2. Execution. Updating the sites ONE AFTER ANOTHER, strictly in place, in a random order,
   with the write-side iolet substitution of the kernels, reproduces the oracle's two-array
   collide-then-propagate populations at even and at odd step counts.

The addresses are written out twice, independently: the read side as the kernels gather
(link q: slot opp(q) of the pull source, slot q of the site itself at a wall), the write side as
the scheme is stated (population q goes to slot q of x + c_q, found through the table row of
opp(q); to slot opp(q) of x itself at a wall).
"""
import numpy as np
import pytest

import oracle
import paper_1906_11925_b200 as hlb
import workloads as W

LATTICES = {"d3q15": hlb.HLB_LATTICE_D3Q15, "d3q19": hlb.HLB_LATTICE_D3Q19}
ORDERS = {"raster": hlb.HLB_ORDER_RASTER, "morton": hlb.HLB_ORDER_MORTON, "tiled": hlb.HLB_ORDER_TILED}

CASES = [  # seed, periodic, shape (nx, ny, nz)
    (0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (20, 5, 4)), (3, 6, (4, 9, 5)),
    (5, 7, (1, 1, 3)), (6, 3, (2, 2, 2)), (7, 0, (12, 11, 10)),
]


def tables(wl, lattice, order):
    flags = LATTICES[lattice] | ORDERS[order]
    t = hlb.hlb_preprocess(wl.site_type, wl.periodic, wl.n_iolets, flags)
    c, w, opp = hlb.hlb_lattice(flags)
    n = t["N"]
    return t["nbr"][:, :n].astype(np.int64), t["canon_of_site"], c, w, opp, n


def read_address(q, i, nbr, opp, n):
    """odd phase: where f_q(x, t) is read -- (slot, site) flattened as slot * n + site"""
    if q == 0:
        return i
    e = nbr[q - 1, i]
    return q * n + i if e < 0 else opp[q] * n + e


def write_address(q, i, nbr, opp, n):
    """odd phase: where f*_q(x, t) is written -- slot q of x + c_q, the pull source of
    direction opp(q); slot opp(q) of x itself when that neighbour is not fluid"""
    if q == 0:
        return i
    e = nbr[opp[q] - 1, i]
    return opp[q] * n + i if e < 0 else q * n + e


@pytest.mark.parametrize("lattice", list(LATTICES))
@pytest.mark.parametrize("order", list(ORDERS))
@pytest.mark.parametrize("seed,periodic,shape", CASES)
def test_read_set_equals_write_set_and_sites_are_disjoint(seed, periodic, shape, order, lattice):
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=3, p_iolet=0.08, periodic=periodic, seed=40 + seed)
    nbr, _, c, w, opp, n = tables(wl, lattice, order)
    nq = len(w)
    owner = np.full(nq * n, -1, dtype=np.int64)
    for i in range(n):
        rd = {read_address(q, i, nbr, opp, n) for q in range(nq)}
        wr = {write_address(q, i, nbr, opp, n) for q in range(nq)}
        assert len(rd) == nq                                  # nq distinct slots
        assert rd == wr, (i, sorted(rd), sorted(wr))          # odd phase: read set = write set
        for a in rd:
            assert owner[a] == -1, f"slot {a} touched by sites {owner[a]} and {i}"
            owner[a] = i
        # even phase: slot q of the site is read, slot opp(q) of the site written
        assert {q * n + i for q in range(nq)} == {opp[q] * n + i for q in range(nq)}
    assert np.all(owner >= 0)                                 # the sites partition all slots


def collide(f, c, w, tau):
    rho = f.sum()
    u = (c * f[:, None]).sum(axis=0) / rho
    cu = c @ u
    feq = w * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * (u @ u))
    return f - (f - feq) / tau, u


def feq_one(q, rho, u, c, w):
    cu = c[q] @ u
    return w[q] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * (u @ u))


def aa_step_in_place(a, odd, nbr, c, w, opp, n, tau, iolet_rho, site_order):
    """One A-A time step on the flat array a[slot * n + site], one site at a time."""
    nq = len(w)
    for i in site_order:
        if odd:
            addr = [read_address(q, i, nbr, opp, n) for q in range(nq)]
        else:
            addr = [q * n + i for q in range(nq)]
        f = np.array([a[x] for x in addr])
        fs, u = collide(f, c, w, tau)
        for p in range(nq):            # out[p] goes where f_p was read: the bounced f*_opp(p) ...
            v = fs[opp[p]]
            if p > 0:
                e = nbr[p - 1, i]
                k = int(e & 0x7fffffff) - 1 if e < 0 else -1
                if k >= 0:             # ... or, on an iolet link, the ghost equilibrium (reading A6)
                    v = feq_one(p, iolet_rho[k], u, c, w)
            a[addr[p]] = v


def gather_state(a, steps, nbr, opp, n, nq):
    """f_q(x, t) after `steps` steps: own slots at even parity, through the table at odd."""
    f = np.empty((n, nq))
    for i in range(n):
        for q in range(nq):
            f[i, q] = a[read_address(q, i, nbr, opp, n)] if steps & 1 else a[q * n + i]
    return f


@pytest.mark.parametrize("lattice", list(LATTICES))
@pytest.mark.parametrize("seed,periodic,shape,order", [
    (0, 0, (7, 6, 5), "raster"), (1, 7, (6, 5, 4), "morton"), (2, 1, (9, 4, 4), "tiled"),
    (5, 7, (1, 1, 3), "raster"), (6, 3, (2, 2, 2), "morton"),
])
def test_sequential_in_place_update_equals_the_oracle(seed, periodic, shape, order, lattice):
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=2, p_iolet=0.08, periodic=periodic,
                       tau=0.6 + 0.05 * seed, seed=70 + seed)
    nbr, canon, c, w, opp, n = tables(wl, lattice, order)
    nq = len(w)
    c = c.astype(np.float64)
    # oracle populations, its own direction order mapped onto the library's by velocity vector
    oc = oracle.velocity_set(lattice)[0]
    col = [int(np.flatnonzero((oc == cq).all(axis=1))[0]) for cq in c.astype(np.int64)]
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, threads=1, lattice=lattice)
    o.set_state(wl.rho0, wl.u0)
    f0 = o.get_populations()[:, col]
    a = np.empty(nq * n)
    for i in range(n):
        for q in range(nq):
            a[q * n + i] = f0[canon[i], q]
    rng = np.random.default_rng(seed)
    for step in range(7):
        got = gather_state(a, step, nbr, opp, n, nq)
        want = o.get_populations()[:, col][canon]
        assert np.max(np.abs(got - want)) < 1e-14, (step, np.max(np.abs(got - want)))
        aa_step_in_place(a, step & 1, nbr, c, w, opp, n, wl.tau, wl.iolet_rho, rng.permutation(n))
        o.step(1)
    o.close()
