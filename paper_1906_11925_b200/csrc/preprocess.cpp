// preprocess.cpp -- geometry preprocessor (host, multi-threaded).
//
// voxel mask -> fluid-site list in the internal order (Morton by default) -> int32
// pull-neighbour table with wall / iolet links encoded as bounce-back targets
// (BASELINE.json north_star (b); "sparse geometries common in
// vascular systems"; the paper's own domains are lists of sites grouped
// in blocks, Table II).
//
// Data structure: the box is cut into 8x8x8 blocks. Every non-empty block keeps a 512-bit
// occupancy map whose bit position is the voxel's rank along the intra-block curve, and
// the index of its first site. Blocks are numbered along a Morton curve over block
// coordinates. With the Morton intra-block curve this is exactly the Morton order of the
// voxel coordinates (the curve is hierarchical), and "which site is voxel (x,y,z)" is
// start[block] + popcount(bits below) -- no dense voxel->site map (17 GB at config 4) and
// no 40-million-key sort.
#include "preprocess.h"

#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cstring>
#include <thread>

#include "../../include/hlb.h"
#include "lattice.h"

namespace hlb {
namespace {

int thread_count() {
  static int n = [] {
    if (const char* e = std::getenv("HLB_THREADS")) {
      int v = std::atoi(e);
      if (v > 0) return v;
    }
    unsigned hc = std::thread::hardware_concurrency();
    return (int)std::min<unsigned>(hc ? hc : 1u, 64u);
  }();
  return n;
}

// fn(begin, end) over [0, n) in chunks of `grain`, dynamically scheduled.
template <class F>
void parallel_for(int64_t n, int64_t grain, F&& fn) {
  if (n <= 0) return;
  const int64_t chunks = (n + grain - 1) / grain;
  const int T = (int)std::min<int64_t>(thread_count(), chunks);
  if (T <= 1) { fn((int64_t)0, n); return; }
  std::atomic<int64_t> next{0};
  auto worker = [&]() {
    for (;;) {
      const int64_t b = next.fetch_add(grain);
      if (b >= n) break;
      fn(b, std::min(n, b + grain));
    }
  };
  std::vector<std::thread> pool;
  pool.reserve(T - 1);
  for (int t = 1; t < T; ++t) pool.emplace_back(worker);
  worker();
  for (auto& th : pool) th.join();
}

inline uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
  v &= 0x1fffffull;
  v = (v | v << 32) & 0x1f00000000ffffull;
  v = (v | v << 16) & 0x1f0000ff0000ffull;
  v = (v | v << 8) & 0x100f00f00f00f00full;
  v = (v | v << 4) & 0x10c30c30c30c30c3ull;
  v = (v | v << 2) & 0x1249249249249249ull;
  return v;
}
inline uint64_t morton3(uint32_t x, uint32_t y, uint32_t z) {
  return spread3(x) | (spread3(y) << 1) | (spread3(z) << 2);
}

struct Slot {          // one non-empty 8x8x8 block
  uint64_t bits[8];    // occupancy by intra-block curve position
  int64_t start;       // internal (base-order) index of its first site
  uint16_t cum[8];     // sites in words below word w
  int64_t block;       // raster block id
  uint64_t key;        // Morton key of the block coordinates
};

struct BlockIndex {
  int nx, ny, nz, nbx, nby, nbz;
  uint16_t pos_of[512];   // ((dz*8+dy)*8+dx) -> curve position
  uint16_t cell_of[512];  // curve position -> ((dz*8+dy)*8+dx)
  std::vector<int32_t> slot_of_block;
  std::vector<Slot> slots;

  inline int64_t lookup(int x, int y, int z) const {
    const int64_t b = ((int64_t)(z >> 3) * nby + (y >> 3)) * nbx + (x >> 3);
    const Slot& s = slots[(size_t)slot_of_block[(size_t)b]];
    const int p = pos_of[((z & 7) << 6) | ((y & 7) << 3) | (x & 7)];
    const int w = p >> 6;
    const uint64_t below = s.bits[w] & ((1ull << (p & 63)) - 1ull);
    return s.start + s.cum[w] + __builtin_popcountll(below);
  }
};

}  // namespace

int preprocess_threads() { return thread_count(); }
void host_parallel_for(int64_t n, int64_t grain, const std::function<void(int64_t, int64_t)>& fn) {
  parallel_for(n, grain, [&](int64_t b, int64_t e) { fn(b, e); });
}

// A group is 32 consecutive sites (one warp). For link q of a group, the lanes whose pull
// source is a fluid site split into runs of lanes with consecutive source indices; with an
// x-fastest site order almost every (group, q) has one to three runs, and 16 bytes then
// replace the 128 bytes of table entries the warp would load.
int64_t build_link_records(const int32_t* nbr, int n_links, int64_t Ns, uint32_t* rec) {
  const int Q = n_links + 1;
  const int64_t G = Ns / 32;
  std::atomic<int64_t> fallback{0};
  parallel_for(G, 1 << 10, [&](int64_t gb, int64_t ge) {
    int64_t fb = 0;
    for (int64_t g = gb; g < ge; ++g) {
      for (int q = 1; q < Q; ++q) {
        const int32_t* e = nbr + (int64_t)(q - 1) * Ns + g * 32;
        uint32_t wall = 0, second = 32, third = 0;  // second / third: lane at which run 1 / run 2 starts
        uint32_t delta[3] = {0u, 0u, 0u};  // source index minus own index (mod 2^32) within a run
        int runs = 0;
        for (int l = 0; l < 32; ++l) {
          if (e[l] < 0) { wall |= 1u << l; continue; }
          const bool cont = l > 0 && e[l - 1] >= 0 && e[l] == e[l - 1] + 1;
          if (!cont) {
            if (runs < 3) delta[runs] = (uint32_t)e[l] - (uint32_t)(g * 32 + l);
            if (runs == 1) second = (uint32_t)l;
            if (runs == 2) third = (uint32_t)l;
            ++runs;
          }
        }
        if (runs < 2) delta[1] = delta[0];
        uint32_t* r = rec + ((size_t)g * (Q - 1) + (size_t)(q - 1)) * 4;
        // a third run: its delta as a 20-bit signed difference to the second run's (consecutive
        // runs of a warp come from neighbouring rows; if it does not fit, the pair is a sentinel)
        const int64_t dd2 = (int64_t)(int32_t)(delta[2] - delta[1]);
        const bool three = runs == 3 && dd2 >= -(1 << 19) && dd2 < (1 << 19);
        if (runs > 3 || (runs == 3 && !three)) {
          r[0] = 0u; r[1] = 0xffffffffu; r[2] = r[3] = 0u;  // sentinel: read the table itself
          ++fb;
        } else {
          r[0] = wall;
          r[1] = three ? (second | 0x40u | (third << 7) | ((uint32_t)(int32_t)dd2 << 12)) : second;
          r[2] = delta[0];
          r[3] = delta[1];
        }
      }
    }
    fallback += fb;
  });
  return fallback.load();
}

int preprocess(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, int n_iolets,
               SiteOrder order, const LatticeDesc& lat, bool count_only, GeometryTables& out,
               std::string& err) {
  const int Q = lat.Q;
  if (!type) { err = "site_type is NULL"; return HLB_EINVAL; }
  if (nx <= 0 || ny <= 0 || nz <= 0) { err = "non-positive box extent"; return HLB_EINVAL; }
  if (n_iolets < 0 || n_iolets > 253) { err = "n_iolets must be in 0..253"; return HLB_EINVAL; }
  if (order != ORDER_MORTON && order != ORDER_RASTER && order != ORDER_TILED) {
    err = "unknown site order"; return HLB_EINVAL;
  }
  BlockIndex bi;
  bi.nx = nx; bi.ny = ny; bi.nz = nz;
  bi.nbx = (nx + 7) >> 3; bi.nby = (ny + 7) >> 3; bi.nbz = (nz + 7) >> 3;
  for (int dz = 0; dz < 8; ++dz)
    for (int dy = 0; dy < 8; ++dy)
      for (int dx = 0; dx < 8; ++dx) {
        const int cell = (dz << 6) | (dy << 3) | dx;
        const int pos = (order == ORDER_TILED) ? cell : (int)morton3(dx, dy, dz);
        bi.pos_of[cell] = (uint16_t)pos;
        bi.cell_of[pos] = (uint16_t)cell;
      }
  const int64_t nblocks = (int64_t)bi.nbx * bi.nby * bi.nbz;
  const int64_t nrows = (int64_t)ny * nz;
  const int max_type = 1 + n_iolets;

  // ---- pass A: occupancy maps per block, fluid count per voxel row, type validation
  const int64_t nbrows = (int64_t)bi.nby * bi.nbz;
  std::vector<std::vector<Slot>> row_slots((size_t)nbrows);
  std::vector<int32_t> row_count((size_t)nrows, 0);
  std::atomic<int> bad_type{0};
  parallel_for(nbrows, 4, [&](int64_t rb, int64_t re) {
    std::vector<uint64_t> acc((size_t)bi.nbx * 8);
    std::vector<uint8_t> touched((size_t)bi.nbx);
    for (int64_t r = rb; r < re; ++r) {
      const int by = (int)(r % bi.nby), bz = (int)(r / bi.nby);
      std::fill(acc.begin(), acc.end(), 0ull);
      std::fill(touched.begin(), touched.end(), (uint8_t)0);
      bool any = false;
      for (int dz = 0; dz < 8; ++dz) {
        const int z = bz * 8 + dz;
        if (z >= nz) break;
        for (int dy = 0; dy < 8; ++dy) {
          const int y = by * 8 + dy;
          if (y >= ny) break;
          const uint8_t* row = type + ((int64_t)z * ny + y) * nx;
          int32_t cnt = 0;
          int x = 0;
          while (x < nx) {
            if (x + 8 <= nx) {  // skip 8 solid voxels at a time
              uint64_t w8;
              std::memcpy(&w8, row + x, 8);
              if (w8 == 0) { x += 8; continue; }
            }
            const int xe = std::min(nx, x + 8);
            for (; x < xe; ++x) {
              const uint8_t t = row[x];
              if (t == 1) {
                const int p = bi.pos_of[(dz << 6) | (dy << 3) | (x & 7)];
                acc[(size_t)(x >> 3) * 8 + (p >> 6)] |= 1ull << (p & 63);
                touched[(size_t)(x >> 3)] = 1;
                any = true;
                ++cnt;
              } else if (t > max_type) {
                bad_type.store(1, std::memory_order_relaxed);
              }
            }
          }
          row_count[(size_t)((int64_t)z * ny + y)] = cnt;
        }
      }
      if (!any) continue;
      auto& dst = row_slots[(size_t)r];
      for (int bx = 0; bx < bi.nbx; ++bx) {
        if (!touched[(size_t)bx]) continue;
        Slot s;
        int c = 0;
        for (int w = 0; w < 8; ++w) {
          s.bits[w] = acc[(size_t)bx * 8 + w];
          s.cum[w] = (uint16_t)c;
          c += __builtin_popcountll(s.bits[w]);
        }
        s.start = c;  // count for now
        s.block = ((int64_t)bz * bi.nby + by) * bi.nbx + bx;
        s.key = morton3((uint32_t)bx, (uint32_t)by, (uint32_t)bz);
        dst.push_back(s);
      }
    }
  });
  if (bad_type.load()) { err = "site type >= 2 + n_iolets"; return HLB_EINVAL; }

  size_t nslots = 0;
  for (auto& v : row_slots) nslots += v.size();
  if (nslots == 0) { err = "no fluid voxel (type 1)"; return HLB_ENOFLUID; }
  bi.slots.reserve(nslots);
  for (auto& v : row_slots) {
    bi.slots.insert(bi.slots.end(), v.begin(), v.end());
    std::vector<Slot>().swap(v);
  }
  std::sort(bi.slots.begin(), bi.slots.end(),
            [](const Slot& a, const Slot& b) { return a.key < b.key; });
  int64_t N = 0;
  for (auto& s : bi.slots) { const int64_t c = s.start; s.start = N; N += c; }
  if (N >= (int64_t)0x7fffffff - 128) { err = "too many fluid sites for int32 indices"; return HLB_ETOOLARGE; }
  out = GeometryTables();
  out.N = N;
  out.Ns = (N + 127) / 128 * 128;
  if (count_only) return HLB_OK;

  bi.slot_of_block.assign((size_t)nblocks, -1);
  for (size_t s = 0; s < bi.slots.size(); ++s) bi.slot_of_block[(size_t)bi.slots[s].block] = (int32_t)s;

  // ---- pass B: voxel of every site in the base (block-curve) order
  std::vector<int64_t> voxel_base((size_t)N);
  parallel_for((int64_t)bi.slots.size(), 64, [&](int64_t sb, int64_t se) {
    for (int64_t si = sb; si < se; ++si) {
      const Slot& s = bi.slots[(size_t)si];
      const int bx = (int)(s.block % bi.nbx), by = (int)((s.block / bi.nbx) % bi.nby),
                bz = (int)(s.block / ((int64_t)bi.nbx * bi.nby));
      int64_t i = s.start;
      for (int w = 0; w < 8; ++w) {
        uint64_t m = s.bits[w];
        while (m) {
          const int p = (w << 6) | __builtin_ctzll(m);
          m &= m - 1;
          const int cell = bi.cell_of[p];
          const int x = bx * 8 + (cell & 7), y = by * 8 + ((cell >> 3) & 7), z = bz * 8 + (cell >> 6);
          voxel_base[(size_t)i++] = ((int64_t)z * ny + y) * nx + x;
        }
      }
    }
  });

  // ---- pass C: canonical rank (ascending voxel index) of every base-order site
  std::vector<int64_t> row_start((size_t)nrows + 1);
  row_start[0] = 0;
  for (int64_t r = 0; r < nrows; ++r) row_start[(size_t)r + 1] = row_start[(size_t)r] + row_count[(size_t)r];
  std::vector<int32_t> canon_base((size_t)N);
  parallel_for(nrows, 256, [&](int64_t rb, int64_t re) {
    for (int64_t r = rb; r < re; ++r) {
      if (row_count[(size_t)r] == 0) continue;
      const int y = (int)(r % ny), z = (int)(r / ny);
      const uint8_t* row = type + r * nx;
      int64_t c = row_start[(size_t)r];
      for (int x = 0; x < nx; ++x)
        if (row[x] == 1) canon_base[(size_t)bi.lookup(x, y, z)] = (int32_t)c++;
    }
  });
  std::vector<int32_t>().swap(row_count);
  std::vector<int64_t>().swap(row_start);

  const bool raster = (order == ORDER_RASTER);
  out.voxel_of_site.resize((size_t)N);
  out.canon_of_site.resize((size_t)N);
  if (raster) {
    parallel_for(N, 1 << 16, [&](int64_t b, int64_t e) {
      for (int64_t i = b; i < e; ++i) {
        const int32_t c = canon_base[(size_t)i];
        out.voxel_of_site[(size_t)c] = voxel_base[(size_t)i];
        out.canon_of_site[(size_t)c] = c;
      }
    });
  } else {
    out.voxel_of_site.swap(voxel_base);
    out.canon_of_site = canon_base;
  }

  // ---- pass D: pull-neighbour table
  const int64_t Ns = out.Ns;
  out.nbr.assign((size_t)(Q - 1) * (size_t)Ns, (int32_t)NBR_WALL_BIT);
  std::vector<uint32_t> iolet_bits((size_t)(Ns / 32), 0u);
  std::atomic<int64_t> n_io_sites{0}, n_wall_links{0};
  const bool px = periodic & 1u, py = periodic & 2u, pz = periodic & 4u;
  parallel_for(N, 1 << 14, [&](int64_t b, int64_t e) {  // grain is a multiple of 32
    int64_t io_sites = 0, wall_links = 0;
    for (int64_t i = b; i < e; ++i) {
      const int64_t v = out.voxel_of_site[(size_t)i];
      const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / ((int64_t)nx * ny));
      bool has_io = false;
      for (int q = 1; q < Q; ++q) {
        int sx = x - lat.c[q][0], sy = y - lat.c[q][1], sz = z - lat.c[q][2];
        bool outside = false;
        if (sx < 0) { if (px) sx += nx; else outside = true; }
        else if (sx >= nx) { if (px) sx -= nx; else outside = true; }
        if (sy < 0) { if (py) sy += ny; else outside = true; }
        else if (sy >= ny) { if (py) sy -= ny; else outside = true; }
        if (sz < 0) { if (pz) sz += nz; else outside = true; }
        else if (sz >= nz) { if (pz) sz -= nz; else outside = true; }
        int32_t entry;
        const uint8_t t = outside ? (uint8_t)0 : type[((int64_t)sz * ny + sy) * nx + sx];
        if (t == 1) {
          const int64_t sb = bi.lookup(sx, sy, sz);
          entry = raster ? canon_base[(size_t)sb] : (int32_t)sb;
        } else if (t == 0) {
          entry = (int32_t)NBR_WALL_BIT;
          ++wall_links;
        } else {
          entry = (int32_t)(NBR_WALL_BIT | (uint32_t)(t - 1));  // iolet k = t-2 -> k+1
          has_io = true;
        }
        out.nbr[(size_t)((q - 1) * Ns + i)] = entry;
      }
      if (has_io) {
        iolet_bits[(size_t)(i >> 5)] |= 1u << (i & 31);
        ++io_sites;
      }
    }
    n_io_sites += io_sites;
    n_wall_links += wall_links;
  });
  out.n_iolet_sites = n_io_sites.load();
  out.n_wall_links = n_wall_links.load();

  // ---- iolet index: {bits, rank} per group and one row of link -> iolet id per flagged site
  const int64_t G = Ns / 32;
  out.iolet_idx.assign((size_t)G * 2, 0u);
  {
    uint32_t rank = 0;
    for (int64_t g = 0; g < G; ++g) {
      out.iolet_idx[(size_t)g * 2] = iolet_bits[(size_t)g];
      out.iolet_idx[(size_t)g * 2 + 1] = rank;
      rank += (uint32_t)__builtin_popcount(iolet_bits[(size_t)g]);
    }
  }
  const int row = iolet_row_bytes(Q);
  out.iolet_links.assign((size_t)(out.n_iolet_sites + 1) * (size_t)row, (uint8_t)0);
  parallel_for(G, 1 << 12, [&](int64_t gb, int64_t ge) {
    for (int64_t g = gb; g < ge; ++g) {
      uint32_t m = iolet_bits[(size_t)g];
      size_t r = out.iolet_idx[(size_t)g * 2 + 1];
      while (m) {
        const int64_t i = g * 32 + __builtin_ctz(m);
        m &= m - 1;
        uint8_t* dst = out.iolet_links.data() + r * (size_t)row;
        for (int q = 1; q < Q; ++q) {
          const uint32_t e = (uint32_t)out.nbr[(size_t)((q - 1) * Ns + i)];
          if ((e & NBR_WALL_BIT) && (e & 0x7fffffffu)) dst[q - 1] = (uint8_t)(e & 0x7fffffffu);  // k + 1
        }
        ++r;
      }
    }
  });

  // ---- pass E: run-length link records
  out.rec.assign((size_t)(Ns / 32) * (Q - 1) * 4, 0u);
  out.n_rec_fallback = build_link_records(out.nbr.data(), Q - 1, Ns, out.rec.data());
  return HLB_OK;
}

void build_bfl_tables(const int32_t* nbr, const int32_t* canon, int Q, int64_t N, int64_t Ns,
                      const double* d27, BflTables& out) {
  const LatticeDesc& lat = lattice_desc(Q == 19);
  out = BflTables();
  std::vector<uint32_t> bits((size_t)(Ns / 32), 0u);
  {
    // threaded over chunks of sites (multiples of 32: a word of `bits` has one writer); the
    // chunks' finds are concatenated in order, so the list is the same for any thread count
    struct Found { std::vector<int32_t> site, behind; std::vector<uint8_t> link; std::vector<double> d; };
    const int64_t grain = 1 << 16;
    const int64_t nchunks = (N + grain - 1) / grain;
    std::vector<Found> found((size_t)nchunks);
    for (int p = 1; p < Q; ++p) {
      // the wall lies along -c_p
      const int idx = (-lat.c[p][2] + 1) * 9 + (-lat.c[p][1] + 1) * 3 + (-lat.c[p][0] + 1);
      const int32_t* e_row = nbr + (size_t)(p - 1) * (size_t)Ns;
      const int32_t* b_row = nbr + (size_t)(opp(p) - 1) * (size_t)Ns;
      host_parallel_for(N, grain, [&](int64_t b, int64_t e) {
        Found& f = found[(size_t)(b / grain)];
        f.site.clear(); f.behind.clear(); f.link.clear(); f.d.clear();
        for (int64_t i = b; i < e; ++i) {
          // a solid-wall link with a fluid site behind the site
          if (e_row[i] != (int32_t)NBR_WALL_BIT || b_row[i] < 0) continue;
          const double dd = d27[(size_t)canon[(size_t)i] * 27 + (size_t)idx];
          if (dd > 0.0 && dd <= 1.0) {
            f.site.push_back((int32_t)i);
            f.behind.push_back(b_row[i]);
            f.link.push_back((uint8_t)p);
            f.d.push_back(dd);
            bits[(size_t)(i >> 5)] |= 1u << (i & 31);
          }
        }
      });
      for (const Found& f : found) {
        out.site.insert(out.site.end(), f.site.begin(), f.site.end());
        out.behind.insert(out.behind.end(), f.behind.begin(), f.behind.end());
        out.link.insert(out.link.end(), f.link.begin(), f.link.end());
        out.d.insert(out.d.end(), f.d.begin(), f.d.end());
      }
    }
  }
  std::vector<int32_t> rank(bits.size());
  for (size_t w = 0; w < bits.size(); ++w) {
    rank[w] = (int32_t)out.n_sites;
    out.n_sites += __builtin_popcount(bits[w]);
  }
  out.nf = (size_t)((out.n_sites + 31) / 32 * 32 + 32);
  out.row = bfl_row_of(Q);
  out.coef.assign(out.row * out.nf, 0.0);
  std::vector<uint32_t> member(out.nf, 0u);
  for (size_t l = 0; l < out.site.size(); ++l) {
    const int64_t i = out.site[l];
    const size_t at = (size_t)rank[(size_t)(i >> 5)] +
                      (size_t)__builtin_popcount(bits[(size_t)(i >> 5)] & ((1u << (i & 31)) - 1u));
    const double dd = out.d[l];
    // one coefficient per opposite pair (2k + 1, 2k + 2) -- its two links are never both
    // interpolated: each needs the site on the other side to be fluid -- and the member word
    const size_t k = (size_t)(out.link[l] - 1) / 2;
    out.coef[at * out.row + k] = dd < 0.5 ? 1.0 - 2.0 * dd : -(1.0 - 1.0 / (2.0 * dd));  // +-(1 - a), kernels.cu
    if ((out.link[l] - 1) & 1) member[at] |= 1u << k;
  }
  for (size_t at = 0; at < out.nf; ++at) {  // the member word sits behind the (Q-1)/2 coefficients of the row
    const uint64_t word = member[at];
    std::memcpy(&out.coef[at * out.row + (size_t)(Q - 1) / 2], &word, sizeof(double));
  }
  out.index.resize(2 * bits.size());
  for (size_t w = 0; w < bits.size(); ++w) {
    out.index[2 * w] = bits[w];
    out.index[2 * w + 1] = (uint32_t)rank[w];
  }
}

}  // namespace hlb
