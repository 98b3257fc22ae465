"""Host logic of the geometry preprocessor (no GPU): brute-force checks of the site
ordering and of the int32 pull-neighbour table on random small masks."""
import numpy as np
import pytest

import paper_1906_11925_b200 as hlb
import workloads as W

C, WT, OPP = hlb.hlb_velocity_set()
WALL = np.int32(-2 ** 31)


def morton_key(x, y, z):
    k = 0
    for b in range(21):
        k |= ((x >> b) & 1) << (3 * b) | ((y >> b) & 1) << (3 * b + 1) | ((z >> b) & 1) << (3 * b + 2)
    return k


LATTICES = {"d3q15": hlb.HLB_LATTICE_D3Q15, "d3q19": hlb.HLB_LATTICE_D3Q19}


def brute_table(st, periodic, vox_of_site, C=C):
    nz, ny, nx = st.shape
    nq = len(C)
    site_of_vox = {int(v): i for i, v in enumerate(vox_of_site)}
    n = len(vox_of_site)
    out = np.zeros((nq - 1, n), dtype=np.int64)
    for i, v in enumerate(vox_of_site):
        x, y, z = int(v % nx), int((v // nx) % ny), int(v // (nx * ny))
        for q in range(1, nq):
            s = [x - int(C[q][0]), y - int(C[q][1]), z - int(C[q][2])]
            outside = False
            for a, ext in enumerate((nx, ny, nz)):
                if s[a] < 0 or s[a] >= ext:
                    if periodic & (1 << a):
                        s[a] %= ext
                    else:
                        outside = True
            t = 0 if outside else int(st[s[2], s[1], s[0]])
            if t == 1:
                out[q - 1, i] = site_of_vox[(s[2] * ny + s[1]) * nx + s[0]]
            elif t == 0:
                out[q - 1, i] = -2 ** 31
            else:
                out[q - 1, i] = -2 ** 31 + (t - 2) + 1
    return out


def test_library_d3q19_set():
    c, w, o = hlb.hlb_lattice(hlb.HLB_LATTICE_D3Q19)
    assert c.shape == (19, 3)
    vecs = {tuple(v) for v in c.tolist()}
    assert len(vecs) == 19 and (0, 0, 0) in vecs
    assert sum(1 for v in vecs if sum(abs(a) for a in v) == 1) == 6
    assert sum(1 for v in vecs if sum(abs(a) for a in v) == 2 and max(abs(a) for a in v) == 1) == 12
    for q in range(19):
        assert np.array_equal(c[o[q]], -c[q]) and o[o[q]] == q
        assert w[q] == {0: 1 / 3, 1: 1 / 18, 2: 1 / 36}[int(c[q] @ c[q])]
    assert abs(w.sum() - 1.0) < 1e-15
    c15, w15, o15 = hlb.hlb_lattice(0)
    assert np.array_equal(c15, C) and np.array_equal(w15, WT) and np.array_equal(o15, OPP)


def test_library_velocity_set_is_d3q15():
    assert {tuple(c) for c in C.tolist()} == {
        (0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
        (1, 1, 1), (-1, -1, -1), (1, 1, -1), (-1, -1, 1), (1, -1, 1), (-1, 1, -1),
        (1, -1, -1), (-1, 1, 1)}
    for q in range(15):
        assert np.array_equal(C[OPP[q]], -C[q]) and OPP[OPP[q]] == q
        assert WT[q] == {0: 2 / 9, 1: 1 / 9, 3: 1 / 72}[int(C[q] @ C[q])]


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("order", [hlb.HLB_ORDER_AUTO, hlb.HLB_ORDER_MORTON, hlb.HLB_ORDER_RASTER,
                                   hlb.HLB_ORDER_TILED])
@pytest.mark.parametrize("seed,periodic,shape", [
    (0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (20, 5, 4)), (3, 2, (4, 19, 5)),
    (4, 4, (5, 4, 17)), (5, 7, (1, 1, 3)), (6, 3, (2, 2, 2)), (7, 0, (16, 16, 16)),
    (8, 5, (17, 9, 23)),
])
def test_table_matches_brute_force(order, seed, periodic, shape, lattice):
    wl = W.random_mask(shape, p_fluid=0.55, n_iolets=3, p_iolet=0.08, periodic=periodic, seed=seed)
    st = wl.site_type
    t = hlb.hlb_preprocess(st, periodic, 3, order | LATTICES[lattice])
    c_lat = hlb.hlb_lattice(LATTICES[lattice])[0]
    assert t["nbr"].shape[0] == len(c_lat) - 1
    canon = wl.fluid_voxels()
    N = len(canon)
    assert t["N"] == N and t["Ns"] % 128 == 0 and N <= t["Ns"] < N + 128
    vox = t["voxel_of_site"]
    assert np.array_equal(np.sort(vox), canon)                       # a permutation of the sites
    assert np.array_equal(canon[t["canon_of_site"]], vox)            # canonical rank is right
    nz, ny, nx = st.shape
    x, y, z = vox % nx, (vox // nx) % ny, vox // (nx * ny)
    if order in (hlb.HLB_ORDER_RASTER, hlb.HLB_ORDER_AUTO):
        assert np.array_equal(vox, canon)
    elif order == hlb.HLB_ORDER_MORTON:
        keys = [morton_key(int(a), int(b), int(c)) for a, b, c in zip(x, y, z)]
        assert keys == sorted(keys)
    else:  # Morton over 8^3 blocks, raster inside
        keys = [(morton_key(int(a) >> 3, int(b) >> 3, int(c) >> 3), int(c) & 7, int(b) & 7, int(a) & 7)
                for a, b, c in zip(x, y, z)]
        assert keys == sorted(keys)
    nbr = t["nbr"]
    assert np.array_equal(nbr[:, :N].astype(np.int64), brute_table(st, periodic, vox, c_lat))
    assert np.all(nbr[:, N:] == WALL)                                 # padding sites: all wall


def test_orders_describe_the_same_links():
    wl = W.by_name("tree", small=True)
    a = hlb.hlb_preprocess(wl.site_type, 0, wl.n_iolets, hlb.HLB_ORDER_MORTON)
    b = hlb.hlb_preprocess(wl.site_type, 0, wl.n_iolets, hlb.HLB_ORDER_RASTER)
    assert a["N"] == wl.n_sites == b["N"]
    # same links, different numbering: map both tables to voxel space and compare
    def links(t):
        N = t["N"]
        nb = t["nbr"][:, :N].astype(np.int64)
        v = t["voxel_of_site"]
        src = np.where(nb >= 0, v[np.clip(nb, 0, N - 1)], nb)
        order = np.argsort(v)
        return src[:, order]
    assert np.array_equal(links(a), links(b))


def test_argument_errors():
    st = np.zeros((3, 3, 3), dtype=np.uint8)
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_preprocess(st, 0, 0, 0)
    assert e.value.code == hlb.HLB_ENOFLUID
    st[1, 1, 1] = 1
    st[0, 0, 0] = 5
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_preprocess(st, 0, 2, 0)                                # type 5 needs 4 iolets
    assert e.value.code == hlb.HLB_EINVAL
    st[0, 0, 0] = 0
    with pytest.raises(hlb.HlbError) as e:
        hlb.hlb_preprocess(st, 0, 0, 0x4000)                           # unknown flag bit
    assert e.value.code == hlb.HLB_EINVAL
    t = hlb.hlb_preprocess(st, 0, 0, 0)                                # isolated site: all walls
    assert t["N"] == 1 and np.all(t["nbr"] == WALL)


# ------------------------------------------------------------------ run-length link records
def decode_records(rec, nbr):
    """Pure-numpy reading of include/hlb.h's record encoding: returns (entries, sentinel)
    with entries[q-1, i] = decoded source index, -1 at wall lanes, and sentinel[g, q-1]."""
    G, NL = rec.shape[0], rec.shape[1]
    out = np.full((NL, G * 32), -1, dtype=np.int64)
    sentinel = np.zeros((G, NL), dtype=bool)
    for g in range(G):
        for k in range(NL):
            wall, second, o0, o1 = (int(v) for v in rec[g, k])
            if second == 0xFFFFFFFF:
                assert wall == 0 and o0 == 0 and o1 == 0
                sentinel[g, k] = True
                continue
            runs_word = second
            second = runs_word & 63
            three = bool(runs_word & 0x40)
            third = (runs_word >> 7) & 31 if three else 32
            dd2 = (runs_word >> 12) - (1 << 20 if runs_word & 0x80000000 else 0)   # 20-bit signed
            assert 1 <= second <= 32
            if three:
                assert second < third <= 31
            else:
                assert runs_word == second                  # no stray bits
            if second == 32:
                assert o1 == o0 and not three
            for l in range(32):
                if (wall >> l) & 1:
                    continue
                off = o1 + dd2 if l >= third else (o1 if l >= second else o0)
                out[k, g * 32 + l] = (off + g * 32 + l) % 2 ** 32
    return out, sentinel


@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("order", [hlb.HLB_ORDER_MORTON, hlb.HLB_ORDER_RASTER, hlb.HLB_ORDER_TILED])
@pytest.mark.parametrize("case", ["random", "random_periodic", "pipe", "tree"])
def test_link_records_decode_to_the_table(order, case, lattice):
    if case == "random":
        wl = W.random_mask((24, 9, 7), p_fluid=0.8, n_iolets=2, p_iolet=0.05, seed=4)
    elif case == "random_periodic":
        wl = W.random_mask((64, 6, 5), p_fluid=1.1, n_iolets=0, periodic=7, seed=5)
    else:
        wl = W.by_name(case, small=True)
    t = hlb.hlb_preprocess(wl.site_type, wl.periodic, wl.n_iolets, order | LATTICES[lattice])
    nbr = t["nbr"].astype(np.int64)
    NL = nbr.shape[0]
    assert NL == {"d3q15": 14, "d3q19": 18}[lattice]
    rec, n_sentinel = hlb.hlb_preprocess_records(t["nbr"])
    assert rec.shape == (t["Ns"] // 32, NL, 4)
    dec, sentinel = decode_records(rec, nbr)
    assert n_sentinel == int(sentinel.sum())
    # brute-force run count per (group, q): <= 2 runs never a sentinel, > 3 runs always, 3 runs
    # a sentinel only if the third delta does not fit
    G = t["Ns"] // 32
    nb = nbr.reshape(NL, G, 32)
    for g in range(G):
        for k in range(NL):
            runs, prev = 0, None
            for l in range(32):
                e = nb[k, g, l]
                if e < 0:
                    prev = None
                    continue
                if prev is None or e != prev + 1:
                    runs += 1
                prev = e
            assert (not sentinel[g, k]) if runs <= 2 else (sentinel[g, k] or runs == 3)
    keep = ~np.repeat(sentinel.T, 32, axis=1)              # [NL, Ns]
    expect = np.where(nbr >= 0, nbr, -1)
    assert np.array_equal(dec[keep], expect[keep])
    if order == hlb.HLB_ORDER_RASTER and case == "random_periodic":
        assert n_sentinel < 0.6 * G * NL                    # x-runs make most records real


def test_link_records_argument_errors():
    with pytest.raises(hlb.HlbError):
        hlb.hlb_preprocess_records(np.zeros((14, 33), dtype=np.int32))
    with pytest.raises(ValueError):
        hlb.hlb_preprocess_records(np.zeros((13, 32), dtype=np.int32))


# ------------------------------------------------------------- interpolated-wall (BFL) tables
@pytest.mark.parametrize("lattice", ["d3q15", "d3q19"])
@pytest.mark.parametrize("seed,periodic,shape", [(0, 0, (7, 6, 5)), (1, 7, (9, 8, 10)), (2, 1, (40, 5, 4)),
                                                 (3, 0, (1, 1, 3)), (4, 5, (37, 9, 6))])
def test_bfl_tables_against_brute_force(seed, periodic, shape, lattice):
    """include/hlb.h, hlb_preprocess_bfl: the per-site rows the step kernels read (one coefficient
    per opposite pair + the member word) decoded back into (site, link) -> coefficient and compared
    with the rule written out link by link from the table, the voxel types and the distances --
    including distances outside (0, 1] (ignored), one-voxel channels (both links of a pair at a
    wall: neither has a fluid site behind, plain bounce-back) and d = 1/2 (coefficient -0.0)."""
    flags = {"d3q15": hlb.HLB_LATTICE_D3Q15, "d3q19": hlb.HLB_LATTICE_D3Q19}[lattice]
    wl = W.random_mask(shape, p_fluid=0.6, n_iolets=2, p_iolet=0.06, periodic=periodic, seed=300 + seed)
    t = hlb.hlb_preprocess(wl.site_type, wl.periodic, wl.n_iolets, flags | hlb.HLB_ORDER_MORTON)
    c, w, opp = hlb.hlb_lattice(flags)
    nq, n, nbr, canon = len(w), t["N"], t["nbr"], t["canon_of_site"]
    rng = np.random.default_rng(seed)
    d27 = rng.uniform(-0.3, 1.3, size=(n, 27))
    d27[rng.random((n, 27)) < 0.1] = 0.5
    got = hlb.hlb_preprocess_bfl(nbr, canon, d27)
    # brute force: link p of site i is interpolated iff its entry is the solid-wall code, the pull
    # source of opp(p) is a fluid site, and 0 < d <= 1
    want = {}
    for i in range(n):
        for p in range(1, nq):
            e, behind = int(nbr[p - 1, i]), int(nbr[opp[p] - 1, i])
            if e >= 0 or (e & 0x7fffffff) != 0 or behind < 0:
                continue
            idx = (1 - c[p][2]) * 9 + (1 - c[p][1]) * 3 + (1 - c[p][0])
            d = d27[canon[i], idx]
            if 0.0 < d <= 1.0:
                want[(i, p)] = 1.0 - 2.0 * d if d < 0.5 else -(1.0 - 1.0 / (2.0 * d))
    assert got["n_interpolated"] == len(want)
    flagged = sorted({i for i, _ in want})
    assert got["n_flagged"] == len(flagged)
    row, pairs = got["coef"].shape[1], (nq - 1) // 2
    assert row == {15: 8, 19: 10}[nq]
    bits, rank = got["index"][:, 0], got["index"][:, 1]
    seen = {}
    for r, i in enumerate(flagged):                      # rows in ascending site order
        g, l = i >> 5, i & 31
        assert (int(bits[g]) >> l) & 1
        assert int(rank[g]) + bin(int(bits[g]) & ((1 << l) - 1)).count("1") == r
        member = int(got["coef"][r, pairs:pairs + 1].view(np.uint64)[0])
        assert member >> pairs == 0
        for k in range(pairs):
            p = 2 * k + 1 + ((member >> k) & 1)
            other = 2 * k + 2 - ((member >> k) & 1)
            assert (i, other) not in want                # never both links of a pair
            cf = got["coef"][r, k]
            if (i, p) in want:
                seen[(i, p)] = cf
            else:
                assert cf == 0.0 and ((member >> k) & 1) == 0
    assert seen.keys() == want.keys()
    for key, cf in want.items():
        assert seen[key] == cf and np.signbit(seen[key]) == np.signbit(cf), key
    # unflagged sites have their bit clear
    mask = np.zeros(t["Ns"], dtype=bool)
    mask[flagged] = True
    unpacked = ((bits[:, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1).astype(bool).ravel()
    assert np.array_equal(unpacked, mask)

