// tlb_step.cu -- the fused force + collide + stream kernel (PAPER Eqs. (1)-(22)) and the
// wall / obstacle boundary kernel (L151, L155, L314), hand-written for sm_100a.
//
// Fused kernel, "strip marching with an asynchronous row pipeline".  A CTA of kW threads owns kW
// lattice columns and marches over a segment of rows.  For every row r one elected thread issues
// 18 bulk asynchronous copies (cp.async.bulk, the 1-D TMA path; SASS UBLKCP) that bring the strip
// of the 18 fluid planes, already shifted in y by the pull rule f_i(x, r) = S_i(x - c_i), into a
// 4-slot ring in shared memory and complete on an mbarrier; the x shift is applied when threads
// read the ring.  Each landed row is used twice without touching HBM or L2 again:
//   (1) when it lands: rho_A, rho_B (Eq. (4)) and psi^s (Eq. (12)) of row r for the strip plus its
//       2-cell halo go into a 6-row ring {rho_A, rho_B, psi^s_A, psi^s_B};
//   (2) two rows later, with stencil rows y-2..y+2 resident: 5x5 force stencils (Eqs. (7), (10),
//       (11)), buoyancy (Eq. (22)), shifted velocities (Eq. (6)), the three BGK collisions
//       (Eqs. (2), (3), (16), (18)) and 27 aligned, coalesced stores of the post-collision
//       populations at (x, y).
// Streaming (Eq. (1)) is the gather of the next step, so stores are never shifted.  The 9 thermal
// planes are only needed in (2) and go straight to registers (LDG issued before the row barrier).
// The four warps of a CTA never meet at a CTA-wide barrier: each warp keeps its own rho / psi ring
// for its 32 columns plus a 2-cell halo (the 4 halo columns are recomputed, not exchanged), waits
// on the mbarrier of the row it needs, and counts itself out of the slot it has finished with; the
// last warp out issues the copy of row r+2 into that slot, a full row of compute ahead of its use.
#include <cstdlib>

#include "tlb_internal.cuh"

namespace tlb {

namespace {

// weights of Fig. 1(b) by |c|^2
__device__ __forceinline__ constexpr double w_c2(int c2) { return c2 == 1 ? 1.0 / 9.0 : (c2 == 2 ? 1.0 / 36.0 : 0.0); }
__device__ __forceinline__ constexpr double p_c2(int c2) {
  return c2 == 1 ? 4.0 / 63.0 : c2 == 2 ? 4.0 / 135.0 : c2 == 4 ? 1.0 / 180.0 : c2 == 5 ? 2.0 / 945.0 : c2 == 8 ? 1.0 / 15120.0 : 0.0;
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

// ---- mbarrier / bulk-copy primitives (PTX; sm_90+ programming model, sm_100a target) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// global -> shared bulk copy of `bytes` (multiple of 16, both sides 16-byte aligned), completing on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
__device__ __forceinline__ double ldg_stream(const double* a, uint64_t policy) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(a), "l"(policy));
  return v;
}
__device__ __forceinline__ void stg_stream(double* a, double v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(a), "d"(v), "l"(policy) : "memory");
}

__device__ __forceinline__ int wrap_row(int r, int ny) {
  r %= ny;
  return r < 0 ? r + ny : r;
}

constexpr int kWarps = kW / 32;
constexpr int kWR = 32 + 4;            // ring columns per warp: its 32 columns and a 2-cell halo each side

struct Smem {
  double f[kSlots][18][kCopyW];              // landed rows of f_A, f_B (columns x0 - kHX .. x0 + kW + kHX - 1)
  double ring[kWarps][kRingRows][4][kWR];    // per warp: rho_A, rho_B, psi^s_A, psi^s_B
  uint8_t flag[kWarps][kRingRows][kWR + 4];  // 1 = solid / wall node
  uint64_t full[kSlots];                     // mbarriers: row landed
  unsigned int done[kSlots];                 // warps that have finished reading the slot (running count)
};

// acq_rel arrive on a shared counter; returns the previous value
__device__ __forceinline__ unsigned int count_out(unsigned int* c) {
  unsigned int old;
  asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(c)) : "memory");
  return old;
}

}  // namespace

// MODE 0: time step (writes Sout).  MODE 1: hydrodynamic fields of the current state.
template <int MODE>
__global__ void __launch_bounds__(kW, 2)
fused_kernel(const Dev d, const double* __restrict__ Sin, double* __restrict__ Sout, int seg_rows,
             double* __restrict__ oRA, double* __restrict__ oRB, double* __restrict__ oUx, double* __restrict__ oUy,
             double* __restrict__ oT) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int nx = d.nx, ny = d.ny, px = d.px;
  const int x0 = blockIdx.x * kW;
  const int x = x0 + t;                       // phase-2 column of this thread
  const int y0 = blockIdx.y * seg_rows;
  const int y1 = min(ny, y0 + seg_rows);
  const long long plane = d.plane;
  const bool periodic = d.periodic_y != 0;
  const uint64_t pol = policy_evict_first();  // every line of Sin is dead once read, Sout until the next step

  if (t == 0) {
#pragma unroll
    for (int s = 0; s < kSlots; s++) { mbar_init(&sm.full[s], 1); sm.done[s] = 0; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // rows are addressed by q = r - (y0 - 2) >= 0: f slot q & 3, ring row q % 6
  const int q_end = (y1 + 2) - (y0 - 2);      // rows r = y0-2 .. y1+1
  auto row_valid = [&](int r) { return periodic || (r >= 0 && r < ny); };
  // elected thread: bring target row r (18 shifted plane rows) into slot q & 3
  auto issue = [&](int q) {
    const int r = y0 - 2 + q;
    if (!row_valid(r)) return;
    const int rr = periodic ? wrap_row(r, ny) : r;
    int rm = rr - 1, rp = rr + 1;             // rows holding the sources of c_y = +1 / -1
    if (periodic) {
      if (rm < 0) rm = ny - 1;
      if (rp >= ny) rp = 0;
    }
    uint64_t* bar = &sm.full[q & 3];
    mbar_expect_tx(bar, 18u * kCopyW * 8u);
    const long long o0 = d.at(x0 - kHX, rr), om = d.at(x0 - kHX, rm), op = d.at(x0 - kHX, rp);
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int i = 0; i < 9; i++) {
        const long long o = cy(i) == 0 ? o0 : (cy(i) > 0 ? om : op);
        bulk_g2s(&sm.f[q & 3][s * 9 + i][0], Sin + (s * 9 + i) * plane + o, kCopyW * 8u, bar, pol);
      }
  };
  if (t == 0)
    for (int q = 0; q < 4 && q < q_end; q++) issue(q);

  // phase-1 columns of this lane within its warp's ring: c = lane (x = x0 + 32 wid - 2 + lane) and,
  // for lane < 4, c = 32 + lane
  const bool extra = lane < kWR - 32;
  const int xw = x0 + 32 * wid - 2;           // lattice column of ring column 0
  auto mask_at = [&](int r, int c) -> uint8_t {
    if (!row_valid(r)) return 1;
    const int rr = periodic ? wrap_row(r, ny) : r;
    return d.solidp[(size_t)rr * px + kXL + xw + c];
  };
  uint8_t m0 = mask_at(y0 - 2, lane), m1 = extra ? mask_at(y0 - 2, 32 + lane) : 1;
  double (*ring)[4][kWR] = sm.ring[wid];
  uint8_t (*flag)[kWR + 4] = sm.flag[wid];

  uint32_t parity = 0;  // one bit per slot
  for (int q = 0; q < q_end; q++) {
    const int r = y0 - 2 + q;
    const int slot = q & 3, rq = q % kRingRows;
    const bool valid = row_valid(r);
    const uint8_t s0 = m0, s1 = m1;
    if (q + 1 < q_end) {  // mask of the next row, a full iteration ahead of its use
      m0 = mask_at(r + 1, lane);
      if (extra) m1 = mask_at(r + 1, 32 + lane);
    }
    // thermal populations of row y = r - 2 (phase 2), issued now, consumed after the force stencil
    const int y = r - 2;
    const bool do2 = y >= y0;
    const bool active = do2 && x < nx;
    double g[9];
    if (active) {
      int ym = y - 1, yp = y + 1;
      if (periodic) {
        if (ym < 0) ym = ny - 1;
        if (yp >= ny) yp = 0;
      }
      const double* g0 = Sin + 18 * plane + d.at(x, y);
      const double* gm = Sin + 18 * plane + d.at(x, ym);
      const double* gp = Sin + 18 * plane + d.at(x, yp);
#pragma unroll
      for (int i = 0; i < 9; i++) {
        const double* b = cy(i) == 0 ? g0 : (cy(i) > 0 ? gm : gp);
        g[i] = ldg_stream(b + i * plane - cx(i), pol);
      }
    }
    // ---- (1) rho, psi of row r (Eqs. (4), (12)); wall values at solid / out-of-domain nodes (L155, R9)
    if (valid) {
      mbar_wait(&sm.full[slot], (parity >> slot) & 1u);
      parity ^= 1u << slot;
    }
#pragma unroll
    for (int pass = 0; pass < 2; pass++) {
      if (pass == 1 && !extra) break;
      const int c = pass == 0 ? lane : 32 + lane;
      const int cf = 32 * wid + c + 2;  // column of the landed rows holding S(x), x = xw + c
      const uint8_t sol = pass == 0 ? s0 : s1;
      double ra = d.rho_wall_A, rb = d.rho_wall_B, pa = d.pss_wall_A, pb = d.pss_wall_B;
      if (!sol) {
        double fa[9], fb[9];
#pragma unroll
        for (int i = 0; i < 9; i++) {
          fa[i] = sm.f[slot][i][cf - cx(i)];
          fb[i] = sm.f[slot][9 + i][cf - cx(i)];
        }
        ra = sum9(fa);
        rb = sum9(fb);
        pa = d.rho0 * (1.0 - exp(-ra * d.inv_rho0));
        pb = d.rho0 * (1.0 - exp(-rb * d.inv_rho0));
      }
      ring[rq][0][c] = ra; ring[rq][1][c] = rb; ring[rq][2][c] = pa; ring[rq][3][c] = pb;
      flag[rq][c] = sol;
    }
    // the 18 fluid populations of (x, y), landed two iterations ago
    double fa[9], fb[9];
    const int slot2 = (q + 2) & 3;  // == (q - 2) & 3
    if (active) {
#pragma unroll
      for (int i = 0; i < 9; i++) {
        fa[i] = sm.f[slot2][i][t + kHX - cx(i)];
        fb[i] = sm.f[slot2][9 + i][t + kHX - cx(i)];
      }
    }
    __syncwarp();  // ring row r of this warp is complete; this warp has read slot2 for the last time
    if (lane == 0 && q >= 2 && (count_out(&sm.done[slot2]) & (kWarps - 1)) == kWarps - 1 && q + 2 < q_end)
      issue(q + 2);  // last warp out: the slot is free
    if (!do2) continue;
    // ---- (2) collide row y = r - 2, whose stencil rows y-2..y+2 = r-4..r are resident
    const int rq0 = (q + kRingRows - 2) % kRingRows;  // ring row of y
    const int cc = lane + 2;                          // ring column of x
    if (active && !flag[rq0][cc]) {
      const double ra = ring[rq0][0][cc], rb = ring[rq0][1][cc], pa = ring[rq0][2][cc], pb = ring[rq0][3][cc];
      // force sums over the 5x5 neighbourhood: cross (w, other species' rho), self (G_a w + G_r p, own psi^s)
      double xAx = 0, xAy = 0, xBx = 0, xBy = 0, sAx = 0, sAy = 0, sBx = 0, sBy = 0;
#pragma unroll
      for (int dy = -2; dy <= 2; dy++) {
        const int sl = (q + kRingRows - 2 + dy) % kRingRows;
#pragma unroll
        for (int dx = -2; dx <= 2; dx++) {
          const int c2 = dx * dx + dy * dy;
          if (c2 == 0) continue;
          const double w = w_c2(c2), p = p_c2(c2);
          const double nsA = ring[sl][2][cc + dx], nsB = ring[sl][3][cc + dx];
          const double kA = d.G11a * w + d.G11r * p, kB = d.G22a * w + d.G22r * p;
          if (dx != 0) { sAx += (kA * dx) * nsA; sBx += (kB * dx) * nsB; }
          if (dy != 0) { sAy += (kA * dy) * nsA; sBy += (kB * dy) * nsB; }
          if (c2 <= 2) {
            const double nrA = ring[sl][0][cc + dx], nrB = ring[sl][1][cc + dx];
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
        const size_t k = (size_t)y * nx + x;
        if (oRA) oRA[k] = ra;
        if (oRB) oRB[k] = rb;
        if (oUx) oUx[k] = uHx;
        if (oUy) oUy[k] = uHy;
        if (oT) oT[k] = T;
      } else {
        collide9(fa, ra, ux + FAx * invA, uy + FAy * invA, d.omega);  // Eq. (6)
        collide9(fb, rb, ux + FBx * invB, uy + FBy * invB, d.omega);
        if (d.thermal) collide9(g, T, uHx, uHy, d.omega_g);           // Eqs. (16), (18)
        double* o = Sout + d.at(x, y);
        const int nsets = d.thermal ? 27 : 18;
#pragma unroll
        for (int i = 0; i < 27; i++)
          if (i < nsets) stg_stream(o + i * plane, i < 9 ? fa[i] : (i < 18 ? fb[i - 9] : g[i - 18]), pol);
        if (x < kGhost || x >= nx - kGhost) {  // periodic images of this column (ghost columns)
          for (int xg = x + nx; xg < nx + kGhost; xg += nx)
#pragma unroll
            for (int i = 0; i < 27; i++)
              if (i < nsets) o[i * plane + (xg - x)] = i < 9 ? fa[i] : (i < 18 ? fb[i - 9] : g[i - 18]);
          for (int xg = x - nx; xg >= -kGhost; xg -= nx)
#pragma unroll
            for (int i = 0; i < 27; i++)
              if (i < nsets) o[i * plane + (xg - x)] = i < 9 ? fa[i] : (i < 18 ? fb[i - 9] : g[i - 18]);
        }
      }
    } else if (MODE == 1 && active) {  // solid site: report the wall values
      const size_t k = (size_t)y * nx + x;
      if (oRA) oRA[k] = d.rho_wall_A;
      if (oRB) oRB[k] = d.rho_wall_B;
      if (oUx) oUx[k] = 0.0;
      if (oUy) oUy[k] = 0.0;
      if (oT) oT[k] = (2 * y < ny) ? d.T_bottom : d.T_top;
    }
  }
}

// Boundary kernel (a9): fills the ghost rows beyond flat walls and the surface of obstacles with the
// values their fluid neighbours will pull, and keeps the ghost columns of those nodes (periodic
// images) valid.  Work items: (node, direction) pairs over 2*nx ghost-row nodes (walls only)
// followed by the n_sites listed solid sites.  For a solid / ghost node s and direction i with
// x = s + c_i fluid:
//   f:  S_i(s) = S_opp(i)(x)                         half-way bounce-back, L151 (R7)
//   g:  S_i(s) = -S_opp(i)(x) + 2 w_i T_w(s)         fixed wall temperature, L314 (R8)
__global__ void __launch_bounds__(256)
boundary_kernel(const Dev d, double* __restrict__ S, const int* __restrict__ sites, int n_sites) {
  const int nx = d.nx, ny = d.ny;
  const int n_ghost = d.periodic_y ? 0 : 2 * nx;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int node = k >> 3, i = (k & 7) + 1;
  if (node >= n_ghost + n_sites) return;
  int sx, sy;  // lattice coordinates of the solid node, sy in -1..ny
  if (node < n_ghost) {
    sx = node < nx ? node : node - nx;
    sy = node < nx ? -1 : ny;
  } else {
    const int s = sites[node - n_ghost];
    sx = s % nx;
    sy = s / nx;
  }
  int x = sx + cx(i), y = sy + cy(i);
  x = x < 0 ? x + nx : (x >= nx ? x - nx : x);
  if (d.periodic_y) y = y < 0 ? y + ny : (y >= ny ? y - ny : y);
  if (y < 0 || y >= ny) return;
  if (d.solid[(size_t)y * nx + x]) return;
  const double Tw = (2 * sy < ny) ? d.T_bottom : d.T_top;
  const long long plane = d.plane;
  const long long os = d.at(sx, sy), ox = d.at(x, y);
  const int io = opp(i);
  const double va = S[io * plane + ox], vb = S[(9 + io) * plane + ox];
  const double vg = d.thermal ? -S[(18 + io) * plane + ox] + 2.0 * wq(i) * Tw : 0.0;
  for (int xg = sx; xg < nx + kGhost; xg += nx) {  // the node and its right-hand images
    S[i * plane + os + (xg - sx)] = va;
    S[(9 + i) * plane + os + (xg - sx)] = vb;
    if (d.thermal) S[(18 + i) * plane + os + (xg - sx)] = vg;
  }
  for (int xg = sx - nx; xg >= -kGhost; xg -= nx) {
    S[i * plane + os + (xg - sx)] = va;
    S[(9 + i) * plane + os + (xg - sx)] = vb;
    if (d.thermal) S[(18 + i) * plane + os + (xg - sx)] = vg;
  }
}

static dim3 strip_grid(const Dev& d, int seg_rows) {
  return dim3((d.nx + kW - 1) / kW, (d.ny + seg_rows - 1) / seg_rows);
}

int configure_kernels() {
  cudaError_t e = cudaFuncSetAttribute(fused_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(fused_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
  return e == cudaSuccess ? 0 : (int)e;
}

// Rows per CTA segment: strips x segments should fill whole waves of 2 CTAs per SM on 148 SMs with
// as few segments as possible (each segment re-reads 4 warm-up rows), never below 16 rows.
int default_seg_rows(int nx, int ny) {
  const int strips = (nx + kW - 1) / kW, slots = 2 * 148;
  int best_seg = ny;
  double best = -1.0;
  for (int waves = 1; waves <= 4; waves++) {
    int segs = waves * slots / strips;
    if (segs < 1) segs = 1;
    int seg = (ny + segs - 1) / segs;
    if (seg < 16) seg = ny < 16 ? ny : 16;
    segs = (ny + seg - 1) / seg;
    const int ctas = strips * segs;
    const int w = (ctas + slots - 1) / slots;
    const double cost = (double)w * (seg + 4);  // rows marched by the busiest slot, incl. warm-up rows
    const double score = (double)ny * strips / slots / cost;  // 1 = perfect
    if (score > best + 1e-9) { best = score; best_seg = seg; }
  }
  return best_seg;
}

int launch_step(const Dev& d, const double* Sin, double* Sout, int seg_rows, cudaStream_t st) {
  fused_kernel<0><<<strip_grid(d, seg_rows), kW, sizeof(Smem), st>>>(d, Sin, Sout, seg_rows, nullptr, nullptr, nullptr,
                                                                     nullptr, nullptr);
  return 1;
}

int launch_fields(const Dev& d, const double* S, double* rhoA, double* rhoB, double* ux, double* uy, double* T,
                  cudaStream_t st) {
  const int seg_rows = default_seg_rows(d.nx, d.ny);
  fused_kernel<1><<<strip_grid(d, seg_rows), kW, sizeof(Smem), st>>>(d, S, nullptr, seg_rows, rhoA, rhoB, ux, uy, T);
  return 1;
}

int launch_boundary(const Dev& d, double* S, const int* sites, int n_sites, cudaStream_t st) {
  const long long n = 8ll * ((d.periodic_y ? 0 : 2 * d.nx) + n_sites);
  if (n == 0) return 0;
  boundary_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, S, sites, n_sites);
  return 1;
}

}  // namespace tlb
