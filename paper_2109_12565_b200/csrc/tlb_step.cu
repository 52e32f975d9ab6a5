// tlb_step.cu -- the fused force + collide + stream kernel (PAPER Eqs. (1)-(22)) and the
// wall / obstacle boundary kernel (L151, L155, L314), hand-written for sm_100a.
//
// Fused kernel, "strip marching": a CTA owns kStripW interior columns plus kHalo halo columns per
// side and marches over a segment of rows.  For every row r it (1) gathers the 18 time-t fluid
// populations f_l,i(x, r) = S_l,i(x - c_i) (pull form, see tlb_internal.cuh), sums rho_A, rho_B
// (Eq. (4)), evaluates psi^s (Eq. (12)) once per site and puts {rho_A, rho_B, psi^s_A, psi^s_B} of the
// row into a kRing-row ring in shared memory; (2) two rows behind, with rows y-2..y+2 resident,
// evaluates the 5x5 force stencils (Eqs. (7), (10), (11)), buoyancy (Eq. (22)), the shifted
// velocities (Eq. (6)), the three BGK collisions (Eqs. (2), (3), (16), (18)) and stores the 27
// post-collision populations at (x, y): aligned, coalesced, one plane row per warp store.
// Streaming (Eq. (1)) is the gather of the next step, so every store is aligned and only loads
// are shifted by one column.  One __syncthreads per row.
#include "tlb_internal.cuh"

namespace tlb {

namespace {

// weights of Fig. 1(b) by |c|^2
__device__ __forceinline__ constexpr double w_c2(int c2) { return c2 == 1 ? 1.0 / 9.0 : (c2 == 2 ? 1.0 / 36.0 : 0.0); }
__device__ __forceinline__ constexpr double p_c2(int c2) {
  return c2 == 1 ? 4.0 / 63.0 : c2 == 2 ? 4.0 / 135.0 : c2 == 4 ? 1.0 / 180.0 : c2 == 5 ? 2.0 / 945.0 : c2 == 8 ? 1.0 / 15120.0 : 0.0;
}

struct RowSrc {  // gather offsets of the 9 directions for one (column, row), in doubles within a plane
  long long o[9];
};

// Source offsets for target (xc, row r): plane i is read at (x - c_ix, r - c_iy).  `r` is an
// in-domain row (0..ny-1); storage row = lattice row + 1 (ghost row below).
__device__ __forceinline__ RowSrc make_src(const Dev& d, int r, int xc, int xm, int xp) {
  int rm = r - 1, rp = r + 1;  // rows holding the sources of c_y = +1 / -1
  if (d.periodic_y) {
    if (rm < 0) rm = d.ny - 1;
    if (rp >= d.ny) rp = 0;
  }
  const long long b0 = (long long)(r + 1) * d.nx, bm = (long long)(rm + 1) * d.nx, bp = (long long)(rp + 1) * d.nx;
  RowSrc s;
  s.o[0] = b0 + xc; s.o[1] = b0 + xm; s.o[2] = bm + xc; s.o[3] = b0 + xp; s.o[4] = bp + xc;
  s.o[5] = bm + xm; s.o[6] = bm + xp; s.o[7] = bp + xp; s.o[8] = bp + xm;
  return s;
}

__device__ __forceinline__ void load9(const double* __restrict__ base, long long plane, const RowSrc& s, double (&f)[9]) {
#pragma unroll
  for (int i = 0; i < 9; i++) f[i] = __ldg(base + i * plane + s.o[i]);
}

__device__ __forceinline__ double sum9(const double (&f)[9]) {  // Eq. (4), same order as written
  double r = f[0];
#pragma unroll
  for (int i = 1; i < 9; i++) r += f[i];
  return r;
}

// BGK relaxation towards the second-order equilibrium, Eqs. (2), (3) (c_s^2 = 1/3)
__device__ __forceinline__ void collide9(double (&f)[9], double dens, double ux, double uy, double omega) {
  const double usq = 1.0 - 1.5 * (ux * ux + uy * uy);
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const double cu = cx(i) * ux + cy(i) * uy;
    const double feq = wq(i) * dens * (usq + 3.0 * cu + 4.5 * cu * cu);
    f[i] = f[i] + omega * (feq - f[i]);
  }
}

}  // namespace

// MODE 0: time step (writes Sout).  MODE 1: hydrodynamic fields of the current state.
template <int MODE>
__global__ void __launch_bounds__(kStripThreads)
fused_kernel(const Dev d, const double* __restrict__ Sin, double* __restrict__ Sout, int seg_rows,
             double* __restrict__ oRA, double* __restrict__ oRB, double* __restrict__ oUx, double* __restrict__ oUy,
             double* __restrict__ oT) {
  __shared__ double ring[kRing][4][kStripThreads];  // [row slot][rho_A, rho_B, psi^s_A, psi^s_B][column]

  const int tx = threadIdx.x;
  const int nx = d.nx, ny = d.ny;
  const int x_raw = blockIdx.x * kStripW - kHalo + tx;
  int xc = x_raw % nx;
  if (xc < 0) xc += nx;
  const int xm = xc == 0 ? nx - 1 : xc - 1;
  const int xp = xc == nx - 1 ? 0 : xc + 1;
  const bool interior = tx >= kHalo && tx < kHalo + kStripW && x_raw < nx;
  const int y0 = blockIdx.y * seg_rows;
  const int y1 = min(ny, y0 + seg_rows);
  const long long plane = d.plane;
  const double* __restrict__ SA = Sin;
  const double* __restrict__ SB = Sin + 9 * plane;
  const double* __restrict__ SG = Sin + 18 * plane;

  int slot = 0;  // ring slot of row r
  for (int r = y0 - 2; r < y1 + 2; r++) {
    // ---- (1) rho, psi of row r (Eqs. (4), (12)); wall values at solid / out-of-domain nodes (L155, R9)
    {
      int rr = r;
      bool wall = false;
      if (d.periodic_y) {
        rr = r % ny;
        if (rr < 0) rr += ny;
      } else if (r < 0 || r >= ny) {
        wall = true;
      }
      double ra = d.rho_wall_A, rb = d.rho_wall_B, pa = d.pss_wall_A, pb = d.pss_wall_B;
      if (!wall && !d.solid[(size_t)rr * nx + xc]) {
        const RowSrc s = make_src(d, rr, xc, xm, xp);
        double fa[9], fb[9];
        load9(SA, plane, s, fa);
        load9(SB, plane, s, fb);
        ra = sum9(fa);
        rb = sum9(fb);
        pa = d.rho0 * (1.0 - exp(-ra * d.inv_rho0));
        pb = d.rho0 * (1.0 - exp(-rb * d.inv_rho0));
      }
      ring[slot][0][tx] = ra; ring[slot][1][tx] = rb; ring[slot][2][tx] = pa; ring[slot][3][tx] = pb;
    }
    __syncthreads();
    // ---- (2) collide row y = r - 2, whose stencil rows y-2..y+2 = r-4..r are resident
    const int y = r - 2;
    if (y >= y0 && interior && !d.solid[(size_t)y * nx + xc]) {
      const RowSrc s = make_src(d, y, xc, xm, xp);
      double fa[9], fb[9], g[9];
      load9(SA, plane, s, fa);
      load9(SB, plane, s, fb);
      load9(SG, plane, s, g);
      const int sl0 = (slot + kRing - 2) % kRing;  // slot of row y
      const double ra = ring[sl0][0][tx], rb = ring[sl0][1][tx], pa = ring[sl0][2][tx], pb = ring[sl0][3][tx];
      // force sums over the 5x5 neighbourhood: cross (w, other species' rho), self (G_a w + G_r p, own psi^s)
      double xAx = 0, xAy = 0, xBx = 0, xBy = 0, sAx = 0, sAy = 0, sBx = 0, sBy = 0;
#pragma unroll
      for (int dy = -2; dy <= 2; dy++) {
        const int sl = (slot + kRing - 2 + dy + kRing) % kRing;
#pragma unroll
        for (int dx = -2; dx <= 2; dx++) {
          const int c2 = dx * dx + dy * dy;
          if (c2 == 0) continue;
          const double w = w_c2(c2), p = p_c2(c2);
          const double nsA = ring[sl][2][tx + dx], nsB = ring[sl][3][tx + dx];
          const double kA = d.G11a * w + d.G11r * p, kB = d.G22a * w + d.G22r * p;
          if (dx != 0) { sAx += (kA * dx) * nsA; sBx += (kB * dx) * nsB; }
          if (dy != 0) { sAy += (kA * dy) * nsA; sBy += (kB * dy) * nsB; }
          if (c2 <= 2) {
            const double nrA = ring[sl][0][tx + dx], nrB = ring[sl][1][tx + dx];
            if (dx != 0) { xAx += (w * dx) * nrB; xBx += (w * dx) * nrA; }
            if (dy != 0) { xAy += (w * dy) * nrB; xBy += (w * dy) * nrA; }
          }
        }
      }
      // Eqs. (7), (8): psi^x = rho / rho0 on both factors
      const double gx = d.G12 * d.inv_rho0 * d.inv_rho0;
      double FAx = -gx * ra * xAx - pa * sAx, FAy = -gx * ra * xAy - pa * sAy;
      double FBx = -gx * rb * xBx - pb * sBx, FBy = -gx * rb * xBy - pb * sBy;
      // moments, Eqs. (5), (17)
      const double T = sum9(g);
      const double jx = (fa[1] - fa[3] + fa[5] - fa[6] - fa[7] + fa[8]) + (fb[1] - fb[3] + fb[5] - fb[6] - fb[7] + fb[8]);
      const double jy = (fa[2] - fa[4] + fa[5] + fa[6] - fa[7] - fa[8]) + (fb[2] - fb[4] + fb[5] + fb[6] - fb[7] - fb[8]);
      // Eq. (22) buoyancy (R12) and the x-acceleration extension
      const double dT = d.thermal ? (T - d.T_ref) : 0.0;
      FAy += ra * d.alpha_g * dT; FBy += rb * d.alpha_g * dT;
      FAx += ra * d.body_ax;      FBx += rb * d.body_ax;
      const double rho = ra + rb;
      const double inv = 1.0 / rho, invA = d.tau / ra, invB = d.tau / rb;
      const double ux = jx * inv, uy = jy * inv;                       // Eq. (5)
      const double uHx = (jx + 0.5 * (FAx + FBx)) * inv, uHy = (jy + 0.5 * (FAy + FBy)) * inv;  // L139
      if (MODE == 1) {
        const size_t k = (size_t)y * nx + xc;
        if (oRA) oRA[k] = ra;
        if (oRB) oRB[k] = rb;
        if (oUx) oUx[k] = uHx;
        if (oUy) oUy[k] = uHy;
        if (oT) oT[k] = T;
      } else {
        collide9(fa, ra, ux + FAx * invA, uy + FAy * invA, d.omega);  // Eq. (6)
        collide9(fb, rb, ux + FBx * invB, uy + FBy * invB, d.omega);
        const long long o = (long long)(y + 1) * nx + xc;
#pragma unroll
        for (int i = 0; i < 9; i++) Sout[i * plane + o] = fa[i];
#pragma unroll
        for (int i = 0; i < 9; i++) Sout[(9 + i) * plane + o] = fb[i];
        if (d.thermal) {
          collide9(g, T, uHx, uHy, d.omega_g);  // Eqs. (16), (18)
#pragma unroll
          for (int i = 0; i < 9; i++) Sout[(18 + i) * plane + o] = g[i];
        }
      }
    } else if (MODE == 1 && y >= y0 && interior) {  // solid site: report the wall values
      const size_t k = (size_t)y * nx + xc;
      if (oRA) oRA[k] = d.rho_wall_A;
      if (oRB) oRB[k] = d.rho_wall_B;
      if (oUx) oUx[k] = 0.0;
      if (oUy) oUy[k] = 0.0;
      if (oT) oT[k] = (2 * y < ny) ? d.T_bottom : d.T_top;
    }
    slot = slot + 1 == kRing ? 0 : slot + 1;
  }
}

// Boundary kernel (a9): fills the ghost rows beyond flat walls and the surface of obstacles with the
// values their fluid neighbours will pull.  Work items: 2*nx ghost nodes (walls only) followed by
// the n_sites listed solid sites.  For a solid / ghost node s and direction i with x = s + c_i fluid:
//   f:  S_i(s) = S_opp(i)(x)                         half-way bounce-back, L151 (R7)
//   g:  S_i(s) = -S_opp(i)(x) + 2 w_i T_w(s)         fixed wall temperature, L314 (R8)
__global__ void __launch_bounds__(128)
boundary_kernel(const Dev d, double* __restrict__ S, const int* __restrict__ sites, int n_sites) {
  const int nx = d.nx, ny = d.ny;
  const int n_ghost = d.periodic_y ? 0 : 2 * nx;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_ghost + n_sites) return;
  int sx, sy;  // lattice coordinates of the solid node, sy in -1..ny
  if (k < n_ghost) {
    sx = k < nx ? k : k - nx;
    sy = k < nx ? -1 : ny;
  } else {
    const int s = sites[k - n_ghost];
    sx = s % nx;
    sy = s / nx;
  }
  const double Tw = (2 * sy < ny) ? d.T_bottom : d.T_top;
  const long long plane = d.plane;
  const long long os = (long long)(sy + 1) * nx + sx;
#pragma unroll
  for (int i = 1; i < 9; i++) {
    int x = sx + cx(i), y = sy + cy(i);
    x = x < 0 ? x + nx : (x >= nx ? x - nx : x);
    if (d.periodic_y) y = y < 0 ? y + ny : (y >= ny ? y - ny : y);
    if (y < 0 || y >= ny) continue;
    if (d.solid[(size_t)y * nx + x]) continue;
    const long long ox = (long long)(y + 1) * nx + x;
    const int io = opp(i);
    S[i * plane + os] = S[io * plane + ox];
    S[(9 + i) * plane + os] = S[(9 + io) * plane + ox];
    if (d.thermal) S[(18 + i) * plane + os] = -S[(18 + io) * plane + ox] + 2.0 * wq(i) * Tw;
  }
}

static dim3 strip_grid(const Dev& d, int seg_rows) {
  return dim3((d.nx + kStripW - 1) / kStripW, (d.ny + seg_rows - 1) / seg_rows);
}

int launch_step(const Dev& d, const double* Sin, double* Sout, int seg_rows, cudaStream_t st) {
  fused_kernel<0><<<strip_grid(d, seg_rows), kStripThreads, 0, st>>>(d, Sin, Sout, seg_rows, nullptr, nullptr, nullptr,
                                                                    nullptr, nullptr);
  return 1;
}

int launch_fields(const Dev& d, const double* S, double* rhoA, double* rhoB, double* ux, double* uy, double* T,
                  cudaStream_t st) {
  const int seg_rows = 64;
  fused_kernel<1><<<strip_grid(d, seg_rows), kStripThreads, 0, st>>>(d, S, nullptr, seg_rows, rhoA, rhoB, ux, uy, T);
  return 1;
}

int launch_boundary(const Dev& d, double* S, const int* sites, int n_sites, cudaStream_t st) {
  const int n = (d.periodic_y ? 0 : 2 * d.nx) + n_sites;
  if (n == 0) return 0;
  boundary_kernel<<<(n + 127) / 128, 128, 0, st>>>(d, S, sites, n_sites);
  return 1;
}

}  // namespace tlb
