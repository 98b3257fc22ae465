// hlb_oracle_dense.cpp -- dense-grid twin of the oracle (pin P9).
//
// TEST INFRASTRUCTURE ONLY (same rule as hlb_oracle.cpp). Written independently of
// hlb_oracle.cpp so that an indexing, wrap or link-classification mistake in either shows
// up as a disagreement on random small masks:
//   * arrays over the WHOLE box (every voxel, fluid or not), no site list, no table;
//   * PUSH form: each fluid voxel collides, then sends f*_q to x + c_q;
//   * its own hand-typed D3Q15 and D3Q19 tables in a different order from hlb_oracle.cpp;
//   * raw populations f_q (the textbook formula verbatim), moments as explicit sums.
//
// Same method: D3Q15 LBGK ("propagation and collision steps"), halfway bounce-back
// ("simple bounce-back"), constant-density iolets:
//   push of f*_q from fluid x to d = x + c_q:
//     d fluid   : f_q(d, t+1)      = f*_q(x, t)
//     d solid   : f_opp(q)(x, t+1) = f*_q(x, t)
//     d iolet k : f_opp(q)(x, t+1) = feq_opp(q)(rho_k, u(x, t))
//     d velocity iolet k (Ladd): f_opp(q)(x, t+1) = f*_q(x, t) - 6 w_q rho(x, t) c_q.u_k
//     d solid with a BFL wall distance wd along c_q and b = x - c_q fluid:
//         wd < 1/2 : f_opp(q)(x, t+1) = 2 wd f*_q(x,t) + (1 - 2 wd) f*_q(b,t)
//         wd >= 1/2: f_opp(q)(x, t+1) = f*_q(x,t)/(2 wd) + (1 - 1/(2 wd)) f*_opp(q)(x,t)
// which is the pull rule of hlb_oracle.cpp read from the other end of the link.

#include <cmath>
#include <cstdint>
#include <vector>

namespace {

struct Lattice {
  int Q;
  const int *CX, *CY, *CZ, *OPP;
  const double* WT;
};

// D3Q15: rest, 6 axis vectors, 8 cube diagonals (hand typed)
const int CX15[15] = {0, 1, -1, 0, 0, 0, 0, 1, 1, 1, 1, -1, -1, -1, -1};
const int CY15[15] = {0, 0, 0, 1, -1, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1};
const int CZ15[15] = {0, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 1, -1};
const int OPP15[15] = {0, 2, 1, 4, 3, 6, 5, 14, 13, 12, 11, 10, 9, 8, 7};
const double WT15[15] = {2.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0,
                         1.0 / 72.0, 1.0 / 72.0, 1.0 / 72.0, 1.0 / 72.0,
                         1.0 / 72.0, 1.0 / 72.0, 1.0 / 72.0, 1.0 / 72.0};

// D3Q19: rest, 6 axis vectors, then the 12 face diagonals plane by plane: xy, xz, yz
// (hand typed; weights 1/3, 1/18, 1/36)
const int CX19[19] = {0, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1, 0, 0, 0, 0};
const int CY19[19] = {0, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1};
const int CZ19[19] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1};
const int OPP19[19] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
const double WT19[19] = {1.0 / 3.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0,
                         1.0 / 18.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
                         1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
                         1.0 / 36.0};

const Lattice L15 = {15, CX15, CY15, CZ15, OPP15, WT15};
const Lattice L19 = {19, CX19, CY19, CZ19, OPP19, WT19};

double feq(const Lattice& L, int q, double rho, double ux, double uy, double uz) {
  double cu = L.CX[q] * ux + L.CY[q] * uy + L.CZ[q] * uz;
  double uu = ux * ux + uy * uy + uz * uz;
  return L.WT[q] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

}  // namespace

extern "C" {

// rho0 / u0: per VOXEL ([nvox], [nvox][3]), read only at fluid voxels; NULL => 1 / 0.
// rho_out / u_out: per voxel, written at fluid voxels, 0 elsewhere.
// Returns 0, or -1 on a bad argument.
static int hlbd_run_impl(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                         int n_iolets, const double* iolet_rho, const uint8_t* iolet_kind,
                         const double* iolet_u, const double* wall_d27, const double* iolet_n,
                         const double* rho0, const double* u0, int64_t steps, double* rho_out,
                         double* u_out, int lattice_q, const double* site_w = nullptr) {
  if (lattice_q != 15 && lattice_q != 19) return -1;
  const Lattice& L = lattice_q == 15 ? L15 : L19;
  const int Q = L.Q;
  const int *CX = L.CX, *CY = L.CY, *CZ = L.CZ, *OPP = L.OPP;
  if (!type || nx <= 0 || ny <= 0 || nz <= 0 || !(tau > 0.5) || steps < 0) return -1;
  const int64_t nvox = (int64_t)nx * ny * nz;
  std::vector<double> f((size_t)nvox * Q, 0.0), g((size_t)nvox * Q, 0.0);
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        const int64_t v = ((int64_t)z * ny + y) * nx + x;
        if (type[v] != 1) continue;
        const double r = rho0 ? rho0[v] : 1.0;
        const double ux = u0 ? u0[v * 3 + 0] : 0.0, uy = u0 ? u0[v * 3 + 1] : 0.0,
                     uz = u0 ? u0[v * 3 + 2] : 0.0;
        for (int q = 0; q < Q; ++q) f[v * Q + q] = feq(L, q, r, ux, uy, uz);
      }
  auto wrap = [&](int& cx_, int& cy_, int& cz_) {  // returns true if outside a non-periodic box
    bool outside = false;
    if (cx_ < 0) { if (periodic & 1u) cx_ += nx; else outside = true; }
    if (cx_ >= nx) { if (periodic & 1u) cx_ -= nx; else outside = true; }
    if (cy_ < 0) { if (periodic & 2u) cy_ += ny; else outside = true; }
    if (cy_ >= ny) { if (periodic & 2u) cy_ -= ny; else outside = true; }
    if (cz_ < 0) { if (periodic & 4u) cz_ += nz; else outside = true; }
    if (cz_ >= nz) { if (periodic & 4u) cz_ -= nz; else outside = true; }
    return outside;
  };
  std::vector<double> fs((size_t)nvox * Q, 0.0), rho_v((size_t)nvox, 0.0), u_v((size_t)nvox * 3, 0.0);
  for (int64_t s = 0; s < steps; ++s) {
    // collision of every fluid voxel
    for (int64_t v = 0; v < nvox; ++v) {
      if (type[v] != 1) continue;
      const double* fv = &f[v * Q];
      double rho = 0.0, jx = 0.0, jy = 0.0, jz = 0.0;
      for (int q = 0; q < Q; ++q) {
        rho += fv[q]; jx += CX[q] * fv[q]; jy += CY[q] * fv[q]; jz += CZ[q] * fv[q];
      }
      const double ux = jx / rho, uy = jy / rho, uz = jz / rho;
      rho_v[v] = rho; u_v[v * 3 + 0] = ux; u_v[v * 3 + 1] = uy; u_v[v * 3 + 2] = uz;
      for (int q = 0; q < Q; ++q) fs[v * Q + q] = fv[q] - (fv[q] - feq(L, q, rho, ux, uy, uz)) / tau;
    }
    // push
    for (int z = 0; z < nz; ++z)
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          const int64_t v = ((int64_t)z * ny + y) * nx + x;
          if (type[v] != 1) continue;
          const double rho = rho_v[v], ux = u_v[v * 3 + 0], uy = u_v[v * 3 + 1], uz = u_v[v * 3 + 2];
          for (int q = 0; q < Q; ++q) {
            const double fstar = fs[v * Q + q];
            int dx = x + CX[q], dy = y + CY[q], dz = z + CZ[q];
            const bool outside = wrap(dx, dy, dz);
            const int64_t d = outside ? -1 : ((int64_t)dz * ny + dy) * nx + dx;
            const int t = outside ? 0 : (int)type[d];
            if (t == 1) g[d * Q + q] = fstar;
            else if (t == 0) {
              // wall along c_q. BFL (linear) if a distance is given and the voxel behind,
              // x - c_q, is fluid; halfway bounce-back otherwise.
              double wd = 0.0;
              if (wall_d27) {
                const double w27 = wall_d27[v * 27 + (CZ[q] + 1) * 9 + (CY[q] + 1) * 3 + (CX[q] + 1)];
                if (w27 > 0.0 && w27 <= 1.0) wd = w27;
              }
              int bx = x - CX[q], by = y - CY[q], bz = z - CZ[q];
              const bool b_out = wrap(bx, by, bz);
              const int64_t b = b_out ? -1 : ((int64_t)bz * ny + by) * nx + bx;
              if (wd > 0.0 && b >= 0 && type[b] == 1) {
                if (wd < 0.5) g[v * Q + OPP[q]] = 2.0 * wd * fstar + (1.0 - 2.0 * wd) * fs[b * Q + q];
                else g[v * Q + OPP[q]] = fstar / (2.0 * wd) + (1.0 - 1.0 / (2.0 * wd)) * fs[v * Q + OPP[q]];
              } else {
                g[v * Q + OPP[q]] = fstar;
              }
            } else {
              if (t - 2 >= n_iolets) return -1;
              const int k = t - 2;
              if (iolet_kind && iolet_kind[k] == 1) {
                // the population leaves along c_q and comes back reversed; seen from the
                // returning direction opp(q) the gain is +6 w rho c_opp(q).u = -6 w rho c_q.u
                const double cu = CX[q] * iolet_u[k * 3 + 0] + CY[q] * iolet_u[k * 3 + 1] +
                                  CZ[q] * iolet_u[k * 3 + 2];
                // site_w: per-voxel weight of the prescribed velocity as seen from this voxel
                g[v * Q + OPP[q]] = fstar - 6.0 * L.WT[q] * rho * ((site_w ? site_w[v] : 1.0) * cu);
              } else if (iolet_n && (iolet_n[k * 3] != 0.0 || iolet_n[k * 3 + 1] != 0.0 || iolet_n[k * 3 + 2] != 0.0)) {
                // normal-projected pressure iolet: only the velocity along the unit normal
                const double len = std::sqrt(iolet_n[k * 3] * iolet_n[k * 3] + iolet_n[k * 3 + 1] * iolet_n[k * 3 + 1] +
                                             iolet_n[k * 3 + 2] * iolet_n[k * 3 + 2]);
                const double n0 = iolet_n[k * 3] / len, n1 = iolet_n[k * 3 + 1] / len, n2 = iolet_n[k * 3 + 2] / len;
                const double un = ux * n0 + uy * n1 + uz * n2;
                g[v * Q + OPP[q]] = feq(L, OPP[q], iolet_rho[k], un * n0, un * n1, un * n2);
              } else {
                g[v * Q + OPP[q]] = feq(L, OPP[q], iolet_rho[k], ux, uy, uz);
              }
            }
          }
        }
    f.swap(g);
  }
  for (int64_t v = 0; v < nvox; ++v) {
    double rho = 0.0, jx = 0.0, jy = 0.0, jz = 0.0;
    if (type[v] == 1) {
      for (int q = 0; q < Q; ++q) {
        const double fq = f[v * Q + q];
        rho += fq; jx += CX[q] * fq; jy += CY[q] * fq; jz += CZ[q] * fq;
      }
      rho_out[v] = rho; u_out[v * 3 + 0] = jx / rho; u_out[v * 3 + 1] = jy / rho; u_out[v * 3 + 2] = jz / rho;
    } else {
      rho_out[v] = 0.0; u_out[v * 3 + 0] = u_out[v * 3 + 1] = u_out[v * 3 + 2] = 0.0;
    }
  }
  return 0;
}

int hlbd_run_lattice(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                     int n_iolets, const double* iolet_rho, const double* rho0, const double* u0,
                     int64_t steps, double* rho_out, double* u_out, int lattice_q) {
  return hlbd_run_impl(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, nullptr, nullptr, nullptr,
                       nullptr, rho0, u0, steps, rho_out, u_out, lattice_q);
}

// iolet_kind [n_iolets]: 0 constant density, 1 Ladd velocity with iolet_u [n_iolets][3];
// wall_d27 per VOXEL [nvox][27]: BFL wall distance along (dx,dy,dz) at (dz+1)*9+(dy+1)*3+(dx+1),
// <= 0 none; NULL: plain bounce-back everywhere.
int hlbd_run_ladd(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                  int n_iolets, const double* iolet_rho, const uint8_t* iolet_kind,
                  const double* iolet_u, const double* rho0, const double* u0, int64_t steps,
                  double* rho_out, double* u_out, int lattice_q) {
  return hlbd_run_impl(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, iolet_kind, iolet_u,
                       nullptr, nullptr, rho0, u0, steps, rho_out, u_out, lattice_q);
}
int hlbd_run_bfl(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                 int n_iolets, const double* iolet_rho, const uint8_t* iolet_kind,
                 const double* iolet_u, const double* wall_d27, const double* rho0,
                 const double* u0, int64_t steps, double* rho_out, double* u_out, int lattice_q) {
  return hlbd_run_impl(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, iolet_kind, iolet_u,
                       wall_d27, nullptr, rho0, u0, steps, rho_out, u_out, lattice_q);
}
// + iolet_n [n_iolets][3]: normals of the constant-density iolets (zero vector: no projection)
int hlbd_run_all(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                 int n_iolets, const double* iolet_rho, const uint8_t* iolet_kind,
                 const double* iolet_u, const double* wall_d27, const double* iolet_n,
                 const double* rho0, const double* u0, int64_t steps, double* rho_out,
                 double* u_out, int lattice_q) {
  return hlbd_run_impl(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, iolet_kind, iolet_u,
                       wall_d27, iolet_n, rho0, u0, steps, rho_out, u_out, lattice_q);
}

// + site_w per VOXEL [nvox]: velocity weight omega(x) of the Ladd links of fluid voxel x
// (NULL: 1 everywhere)
int hlbd_run_weights(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
                     int n_iolets, const double* iolet_rho, const uint8_t* iolet_kind,
                     const double* iolet_u, const double* wall_d27, const double* iolet_n,
                     const double* site_w, const double* rho0, const double* u0, int64_t steps,
                     double* rho_out, double* u_out, int lattice_q) {
  return hlbd_run_impl(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, iolet_kind, iolet_u,
                       wall_d27, iolet_n, rho0, u0, steps, rho_out, u_out, lattice_q, site_w);
}

int hlbd_run(const uint8_t* type, int nx, int ny, int nz, unsigned periodic, double tau,
             int n_iolets, const double* iolet_rho, const double* rho0, const double* u0,
             int64_t steps, double* rho_out, double* u_out) {
  return hlbd_run_lattice(type, nx, ny, nz, periodic, tau, n_iolets, iolet_rho, rho0, u0, steps,
                          rho_out, u_out, 15);
}

}  // extern "C"
