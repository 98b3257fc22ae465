// preprocess.h -- geometry preprocessor (host): voxel mask -> ordered site list + int32
// pull-neighbour table. Subsystem (b) of BASELINE.json north_star; SURVEY.md §8(a) row S0.
#pragma once
#include <cstdint>
#include <functional>
#include <string>
#include <vector>

#include "lattice.h"

namespace hlb {

enum SiteOrder { ORDER_MORTON = 0, ORDER_RASTER = 1, ORDER_TILED = 2 };

struct GeometryTables {
  int64_t N = 0;    // fluid sites
  int64_t Ns = 0;   // plane stride of every [slot][site] array: N rounded up to 128
  std::vector<int64_t> voxel_of_site;  // [N]  internal order -> linear voxel index
  std::vector<int32_t> canon_of_site;  // [N]  internal order -> canonical rank
  std::vector<int32_t> nbr;            // [Q-1][Ns], encoding: include/hlb.h
  // Iolet index (the only thing the step kernels read about iolets): per group of 32 sites
  // {bits, rank}: bit (i & 31) of bits = site i has an iolet link; rank = number of such sites
  // in the groups below. Site i's links are row rank + popcount(bits below lane i & 31) of
  // iolet_links: byte p - 1 of the row = k + 1 if pull link p crosses iolet k, else 0.
  std::vector<uint32_t> iolet_idx;     // [Ns/32][2]
  std::vector<uint8_t> iolet_links;    // [n_iolet_sites + 1][iolet_row_bytes(Q)]
  std::vector<uint32_t> rec;           // [Ns/32][Q-1][4] run-length link records (include/hlb.h)
  int64_t n_rec_fallback = 0;          // (group, q) pairs with more than 2 runs (record = sentinel)
  int64_t n_iolet_sites = 0;
  int64_t n_wall_links = 0;
};

// Returns 0 or a negative hlb_status; `err` gets the message. With count_only the tables
// are left empty and only N / Ns are set.
int preprocess(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, int n_iolets,
               SiteOrder order, const LatticeDesc& lat, bool count_only, GeometryTables& out,
               std::string& err);

// Run-length link records of a finished table: rec [Ns/32][Q-1][4] (encoding: include/hlb.h,
// hlb_preprocess_records). Returns the number of (group, q) pairs that got the sentinel.
int64_t build_link_records(const int32_t* nbr, int n_links, int64_t Ns, uint32_t* rec);

// Bytes of one row of GeometryTables::iolet_links: Q - 1 bytes rounded up to 16 (one or two
// 128-bit loads).
inline int iolet_row_bytes(int Q) { return (Q - 1 + 15) / 16 * 16; }

int preprocess_threads();

// fn(begin, end) over [0, n) in chunks of `grain`, dynamically scheduled on the preprocessor's
// host threads (HLB_THREADS, else the hardware concurrency); also used by the set-up calls of
// the API that loop over all sites.
// Interpolated-wall (BFL) tables, built from the pull table and the wall distances
// (hlb_set_wall_distance; include/hlb.h, hlb_preprocess_bfl). A link p of site i is
// interpolated when its table entry is a solid wall, the site behind (the pull source of
// opp(p)) is fluid, and 0 < d <= 1 is given for it.
struct BflTables {
  // every interpolated link, link-major (all of direction 1, then 2, ...; sites ascending)
  std::vector<int32_t> site, behind;
  std::vector<uint8_t> link;
  std::vector<double> d;
  // site form for the step kernels (BflFused in kernels.cuh)
  std::vector<uint32_t> index;  // [Ns/32][2] {bits, rank}
  std::vector<double> coef;     // [nf][row]
  int64_t n_sites = 0;          // sites with at least one interpolated link
  size_t row = 0, nf = 0;       // doubles per row; rows allocated (n_sites rounded up + 32)
};
inline size_t bfl_row_of(int Q) { return (size_t)(((Q - 1) / 2 + 2) / 2 * 2); }
void build_bfl_tables(const int32_t* nbr, const int32_t* canon, int Q, int64_t N, int64_t Ns,
                      const double* d27, BflTables& out);

void host_parallel_for(int64_t n, int64_t grain, const std::function<void(int64_t, int64_t)>& fn);

}  // namespace hlb
