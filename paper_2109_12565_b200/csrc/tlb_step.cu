// tlb_step.cu -- the fused force + collide + stream kernel (PAPER Eqs. (1)-(22)) and the
// wall / obstacle boundary kernel (L151, L155, L314), hand-written for sm_100a.
//
// Fused kernel, "strip marching with an asynchronous row pipeline".  A CTA of 2 kW threads (two per
// lattice column, one per species) owns kW columns and marches over a segment of rows.  For every row r one elected thread issues
// ONE tensor-map copy (cp.async.bulk.tensor.5d, TMA; SASS UTMALDG) whose box holds the strip of all 18 fluid
// planes, each already shifted in y by the pull rule f_i(x, r) = S_i(x - c_i) (the planes are stored in c_y
// order so that the shift is a stride of the tensor map, tlb_internal.cuh), into a 4-slot ring in shared
// memory, completing on an mbarrier; the x shift is applied when threads read the ring.  (The
// two wrap rows of a y-periodic lattice use 18 1-D bulk copies, SASS UBLKCP, instead.)  Each landed row is
// used twice without touching HBM or L2 again:
//   (1) when it lands: rho_A, rho_B (Eq. (4)) and psi^s (Eq. (12)) of row r for the strip plus its
//       2-cell halo go into a 6-row ring {rho_A, rho_B, psi^s_A, psi^s_B};
//   (2) two rows later, with stencil rows y-2..y+2 resident: 5x5 force stencils (Eqs. (7), (10),
//       (11)), buoyancy (Eq. (22)), shifted velocities (Eq. (6)), the three BGK collisions
//       (Eqs. (2), (3), (16), (18)) and 27 aligned, coalesced stores of the post-collision
//       populations at (x, y).
// Streaming (Eq. (1)) is the gather of the next step, so stores are never shifted.  The 9 thermal
// planes are only needed in (2) and go straight to registers (LDG issued before the row barrier).
// The eight warps of a CTA never meet at a CTA-wide barrier: each warp keeps its own rho / psi ring
// for its 16 columns plus a 2-cell halo (the 4 halo columns are recomputed, not exchanged), waits
// on the "full" mbarrier of the row it needs and arrives on the "empty" mbarrier of the slot it has
// finished with; the warps take turns re-arming the slots, each at the top of an iteration and with a
// slot that the others left an iteration earlier, so that the issuing warp does not wait.
// tau = 1 (the paper's Table A.3, every BASELINE config) has its own instantiation: see Smem.
#include "tlb_internal.cuh"

namespace tlb {

namespace {

// weights of Fig. 1(b) by |c|^2
__device__ __forceinline__ constexpr double w_c2(int c2) { return c2 == 1 ? 1.0 / 9.0 : (c2 == 2 ? 1.0 / 36.0 : 0.0); }
__device__ __forceinline__ constexpr double p_c2(int c2) {
  return c2 == 1 ? 4.0 / 63.0 : c2 == 2 ? 4.0 / 135.0 : c2 == 4 ? 1.0 / 180.0 : c2 == 5 ? 2.0 / 945.0 : c2 == 8 ? 1.0 / 15120.0 : 0.0;
}

__device__ __forceinline__ double sum9(const double (&f)[9]) {  // Eq. (4); pairwise: depth 4 instead of 8
  return (((f[0] + f[1]) + (f[2] + f[3])) + ((f[4] + f[5]) + (f[6] + f[7]))) + f[8];
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
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)  // suspend-time hint: sleep in hardware instead of spinning
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
// tensor-map copy (TMA, SASS UTMALDG) of the box at coordinates (c0 .. c4) of a 5-D map, completing on `bar`
__device__ __forceinline__ void tma_g2s_5d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4,
                                           uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7], %8;" ::"r"(smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
// L2 prefetch of the box at (c0 .. c3) of a 4-D map (SASS UTMAPF)
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];" ::"l"(map), "r"(c0), "r"(c1),
               "r"(c2), "r"(c3)
               : "memory");
}
// L2 prefetch of `bytes` (multiple of 16, 16-byte aligned): starts the HBM read rows ahead of the loads that use it
__device__ __forceinline__ void prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(__cvta_generic_to_global(src)), "r"(bytes) : "memory");
}
// (L1 may keep the line: the x-shifted loads of neighbouring lanes and warps touch every line twice; measured -1.6 %
// sustained against L1::no_allocate)
__device__ __forceinline__ double ldg_stream(const double* a, uint64_t policy) {
  double v;
  asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(a), "l"(policy));
  return v;
}
__device__ __forceinline__ double ldg_stream(const float* a, uint64_t policy) {
  float v;
  asm volatile("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(a), "l"(policy));
  return (double)v;
}
__device__ __forceinline__ void stg_stream(double* a, double v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(a), "d"(v), "l"(policy) : "memory");
}
__device__ __forceinline__ void stg_stream(float* a, double v, uint64_t policy) {
  asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(a), "f"((float)v), "l"(policy) : "memory");
}

// e^x for x <= 0 (the argument of Eq. (12) is -rho / rho0): Cody-Waite reduction x = k ln2 + r,
// |r| <= ln2 / 2, degree-12 Taylor polynomial (truncation < 2e-16 relative) in Estrin form (short
// dependency chains), exponent add.  Arguments below -700 are clamped (e^-700 ~ 1e-304 is far below
// one ulp of the 1 in 1 - e^x).  No special cases: about half the instructions of the library exp,
// within 1 ulp of it on this range.
__device__ __forceinline__ double exp_nonpos(double x) {
  x = fmax(x, -700.0);
  const double shifter = 6755399441055744.0;  // 1.5 * 2^52: the integer part lands in the low word
  const double t = fma(x, 1.4426950408889634074, shifter);
  const int k = __double2loint(t);
  const double kf = t - shifter;
  double r = fma(kf, -6.93147180369123816490e-01, x);
  r = fma(kf, -1.90821492927058770002e-10, r);
  const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
  const double a01 = fma(r, 1.0, 1.0), a23 = fma(r, 1.0 / 6.0, 0.5), a45 = fma(r, 1.0 / 120.0, 1.0 / 24.0),
               a67 = fma(r, 1.0 / 5040.0, 1.0 / 720.0), a89 = fma(r, 1.0 / 362880.0, 1.0 / 40320.0),
               aab = fma(r, 1.0 / 39916800.0, 1.0 / 3628800.0);
  const double b0 = fma(r2, a23, a01), b1 = fma(r2, a67, a45), b2 = fma(r2, aab, a89);
  const double c0 = fma(r4, b1, b0), c1 = fma(r4, 1.0 / 479001600.0, b2);
  const double p = fma(r8, c1, c0);
  return __hiloint2double(__double2hiint(p) + (k << 20), __double2loint(p));
}

// 1 / a for normal a > 0: hardware seed (20 bits) and two Newton steps; within 1 ulp, no slow path
__device__ __forceinline__ double rcp_pos(double a) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  double e = fma(-a, y, 1.0);
  y = fma(y, e, y);
  e = fma(-a, y, 1.0);
  y = fma(y, e, y);
  return y;
}

__device__ __forceinline__ int wrap_row(int r, int ny) {
  r %= ny;
  return r < 0 ? r + ny : r;
}

// The thermal populations reach the lanes through plain loads issued in the iteration that uses them, so their
// latency is exposed unless the lines are already in L2: the warp that re-arms a slot also prefetches (one
// cp.async.bulk.prefetch.tensor.4d, SASS UTMAPF) the 9 thermal plane rows of the row that reaches phase 2
// kGPrefetchRows iterations later (measured on config 4, same box:
// 0.717 ms without, 0.724 / 0.695 / 0.684 / 0.682 / 0.684 / 0.690 / 0.714 ms at 1 / 2 / 3 / 4 / 6 / 8 / 12 rows;
// prefetching the 18 fluid plane rows as well costs 5 %: the bulk copies already run a row and a half ahead).
constexpr int kGPrefetchRows = 4;
constexpr int kCtasPerSM = 256 / kW;     // shared memory allows 2 CTAs of 128 columns (or 1 of 256) per SM
constexpr int kThreads = 2 * kW;       // two threads per lattice column: lane 2k = species A, 2k+1 = species B
constexpr int kWarps = kThreads / 32;  // 8
constexpr int kWC = 16;                // lattice columns per warp
constexpr int kWR = kWC + 4;           // ring columns per warp: its 16 columns and a 2-cell halo each side

// ST = storage type of the populations (double, or float for the pop_precision = 32 bandwidth study; the
// arithmetic is fp64 either way).  Row stride of the landed rows in shared memory: kCopyW doubles, or
// kCopyW + 8 floats so that the two species of a lane pair fall into disjoint banks.
template <typename ST> struct SlotW { static constexpr int v = kCopyW; };
template <> struct SlotW<float> { static constexpr int v = kCopyW + 8; };

// TAU1 (tau = 1, the time step only): the collision needs rho_l, j and F of a site, not its populations, so phase 1
// also leaves the momentum of its row in a small ring and a landed row is dead after phase 1: 3 slots instead of 4,
// and phase 2 reads one 16-byte pair instead of 9 populations.  Phase 2 then runs THREE rows behind phase 1, so that
// inside one iteration the two phases touch disjoint ring rows and are independent: they sit in one basic block
// (phase 1 is branch-free there) and the compiler interleaves their dependency chains.
template <typename ST, bool TAU1>
struct Smem {
  static constexpr int kS = TAU1 ? 3 : kSlots;
  ST f[kS][18][SlotW<ST>::v];                // landed rows of f_A, f_B (columns x0 - kHX .. x0 + kW + kHX - 1)
  double2 jr[TAU1 ? kWarps : 1][TAU1 ? 4 : 1][kWC][2];  // TAU1: per warp, 4 rows of {j_x, j_y} of (column, species)
  double rho[kWarps][kRingRows][kWR][2];     // per warp: {rho_A, rho_B} per column (a lane pair reads 16 contiguous bytes,
  double psi[kWarps][kRingRows][kWR][2];     //           {psi^s_A, psi^s_B}          a half-warp 128: conflict-free)
  uint8_t flag[kWarps][kRingRows][kWR + 4];  // 1 = solid / wall node
  uint64_t full[kSlots];                     // mbarriers: row landed
  uint64_t empty[kSlots];                    // mbarriers: all kWarps warps have finished reading the slot
  uint32_t ticket[kSlots];                   // general tau: arrivals per slot so far (elects the warp that re-arms it)
};

// release arrive of one thread on an mbarrier (the warp is done with the slot the barrier guards)
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// Election of the warp that re-arms a slot: a plain shared counter per slot, bumped by lane 0 of every warp AFTER its
// arrive on the slot's "empty" barrier.  The warp that sees kWarps - 1 (mod kWarps) knows the other arrivals have been
// made, so its acquiring wait on "empty" (below, before the copy is issued) falls through at once.
__device__ __forceinline__ uint32_t slot_ticket(uint32_t* cnt) {
  uint32_t old;
  asm volatile("atom.relaxed.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(cnt)) : "memory");
  return old;
}
__device__ __forceinline__ double pair(double v) { return __shfl_xor_sync(0xffffffffu, v, 1); }  // the other species' lane

// BGK relaxation of one population towards the second-order equilibrium, Eqs. (2), (3) (c_s^2 = 1/3);
// cu = c_i . u, usq = 1 - 1.5 |u|^2, owd = omega * w_i * density, om1 = 1 - omega:
// f - (f - f_eq) / tau  =  (1 - omega) f + omega f_eq
__device__ __forceinline__ double relax(double f, double owd, double cu, double usq, double om1) {
  return om1 * f + owd * (usq + 3.0 * cu + 4.5 * cu * cu);
}
// the same for tau = 1 (omega = 1, every BASELINE config): the population relaxes onto its equilibrium and
// (1 - omega) f = 0 exactly, so the result is bit-identical to relax() with one multiply less
__device__ __forceinline__ double relax_tau1(double owd, double cu, double usq) {
  return owd * (usq + 3.0 * cu + 4.5 * cu * cu);
}

}  // namespace

// MODE 0: time step (writes Sout).  MODE 1: hydrodynamic fields of the current state.  MODE 2: the stress
// field P_xy (reading R21).  MODE 3: per-CTA partial sums of the observables (a10), reduced in the same pass.
// Work split inside a lane pair (s = lane & 1): lane s owns species s -- its density and psi^s
// (phase 1), its force, shifted velocity, collision and 9 stores (phase 2) -- and half of the thermal
// set: s = 0 takes g_0, g_1, g_2, g_5, g_6, s = 1 the opposite directions g_3, g_4, g_7, g_8, so both
// lanes run the same code on (c_i, u) and (-c_i, -u).  Partial sums (j, F, T) cross by one shuffle.
template <int MODE, bool PERIODIC, typename ST, bool TAU1>
__global__ void __launch_bounds__(kThreads, kCtasPerSM)
fused_kernel(const Dev d, const ST* __restrict__ Sin, ST* __restrict__ Sout, int seg_rows, int ya, int yb,
             const FusedOut out, const __grid_constant__ TMaps tm) {
  constexpr bool kTensor = true;  // tensor-map row copies (1-D bulk copies remain for the two wrap rows of a y-periodic lattice)
  double* __restrict__ const oRA = out.rhoA;
  double* __restrict__ const oRB = out.rhoB;
  double* __restrict__ const oUx = out.ux;
  double* __restrict__ const oUy = out.uy;
  double* __restrict__ const oT = out.T;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using SmemT = Smem<ST, TAU1>;
  SmemT& sm = *reinterpret_cast<SmemT*>(smem_raw);
  constexpr int kSW = SlotW<ST>::v, kB = (int)sizeof(ST), kS = SmemT::kS;
  static_assert(!TAU1 || MODE == 0, "the tau = 1 path is the time step only");
  auto slot_of = [](int q) { return TAU1 ? q % 3 : q & 3; };

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int k = lane >> 1, s = lane & 1;
  const int nx = d.nx, ny = d.ny, px = d.px;
  const int x0 = blockIdx.x * kW;
  const int xw = x0 + kWC * wid - 2;          // lattice column of this warp's ring column 0
  const int x = xw + 2 + k;                   // phase-2 column of this lane pair
  const int y0 = ya + blockIdx.y * seg_rows;  // this CTA marches rows [y0, y1) of the launch's range [ya, yb)
  const int y1 = min(yb, y0 + seg_rows);
  const long long plane = d.plane;
  const long long planeB = plane * kB, rowB = d.row * kB;
  const uint64_t pol = policy_evict_first();  // every line of Sin is dead once read, Sout until the next step

  if (t == 0) {
#pragma unroll
    for (int i = 0; i < kS; i++) { mbar_init(&sm.full[i], 1); mbar_init(&sm.empty[i], kWarps); sm.ticket[i] = 0; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // rows are addressed by q = r - (y0 - 2) >= 0: f slot q & 3, ring row q % 6
  const int q_end = (y1 + 2) - (y0 - 2);      // rows r = y0-2 .. y1+1
  auto row_valid = [&](int r) { return PERIODIC || (r >= 0 && r < ny); };
  // elected lane: bring target row r (18 shifted plane rows) into slot q & 3
  auto issue = [&](int q) {
    const int r = y0 - 2 + q;
    if (!row_valid(r)) return;
    const int rr = PERIODIC ? wrap_row(r, ny) : r;
    int rm = rr - 1, rp = rr + 1;             // rows holding the sources of c_y = +1 / -1
    if (PERIODIC) {
      if (rm < 0) rm = ny - 1;
      if (rp >= ny) rp = 0;
    }
    const int sl = slot_of(q);
    uint64_t* bar = &sm.full[sl];
    if (kTensor && (!PERIODIC || (rr > 0 && rr < ny - 1))) {
      // one copy: box kSW x 1 x 3 x 3 x 2 = the 18 fluid plane rows, each shifted by its c_y (tlb_internal.cuh); kSW is
      // the row pitch of a slot (136 doubles; 144 floats: the padding columns are fetched too, they exist in the buffer)
      mbar_expect_tx(bar, 18u * kSW * kB);
      tma_g2s_5d(&sm.f[sl][0][0], &tm.f, kXL + x0 - kHX, rr, 0, 0, 0, bar, pol);
      return;
    }
    mbar_expect_tx(bar, 18u * kCopyW * kB);
    const long long o0 = d.at(x0 - kHX, rr), om = d.at(x0 - kHX, rm), op = d.at(x0 - kHX, rp);
#pragma unroll
    for (int l = 0; l < 2; l++)
#pragma unroll
      for (int i = 0; i < 9; i++) {
        const long long o = cy(i) == 0 ? o0 : (cy(i) > 0 ? om : op);
        bulk_g2s(&sm.f[sl][l * 9 + pslot(i)][0], Sin + (l * 9 + pslot(i)) * plane + o, kCopyW * kB, bar, pol);
      }
  };
  if (t == 0) {
    for (int q = 0; q < (TAU1 ? 1 : kS) && q < q_end; q++) issue(q);
  }

  // phase-1 tasks of this lane: ring column k and, for lanes < 8, ring column 16 + k; species s
  const bool extra = lane < 2 * (kWR - kWC);
  auto mask_at = [&](int r, int c) -> uint8_t {
    if (!row_valid(r)) return 1;
    const int rr = PERIODIC ? wrap_row(r, ny) : r;
    return d.solidp[(size_t)rr * px + kXL + xw + c];
  };
  uint8_t m0 = mask_at(y0 - 2, k), m1 = extra ? mask_at(y0 - 2, kWC + k) : 1;
  double (*rho_r)[kWR][2] = sm.rho[wid];
  double (*psi_r)[kWR][2] = sm.psi[wid];
  uint8_t (*flag)[kWR + 4] = sm.flag[wid];

  // per-lane constants: own wall values, own self-interaction stencil coefficients G^a w + G^r p by |c|^2
  const double rho_wall = s ? d.rho_wall_B : d.rho_wall_A, pss_wall = s ? d.pss_wall_B : d.pss_wall_A;
  const double Ga = s ? d.G22a : d.G11a, Gr = s ? d.G22r : d.G11r;
  const double k1 = Ga * w_c2(1) + Gr * p_c2(1), k2 = Ga * w_c2(2) + Gr * p_c2(2), k4 = Ga * w_c2(4) + Gr * p_c2(4),
               k5 = Ga * w_c2(5) + Gr * p_c2(5), k8 = Ga * w_c2(8) + Gr * p_c2(8);
  const double k4d = 2.0 * k4, k5d = 2.0 * k5, k8d = 2.0 * k8;
  const double gx = d.G12 * d.inv_rho0 * d.inv_rho0;  // Eqs. (7), (8): psi^x = rho / rho0 on both factors
  const double om1 = 1.0 - d.omega, om1g = 1.0 - d.omega_g;
  const double sgn = s ? -1.0 : 1.0;                  // this lane's thermal directions are sgn * {c_1, c_2, c_5, c_6}

  // running byte pointers of row y = y0 (advanced by one row per phase-2 iteration)
  // thermal planes of lane s (internal order pslot()): g_0 at plane 3 (lane 0 only), g_1 / g_3 at 4 + s,
  // {g_2, g_5, g_6} at 0, 1, 2 (lane 0), {g_4, g_7, g_8} at 6, 7, 8 (lane 1): 6 planes higher
  const char* gp = reinterpret_cast<const char*>(Sin + (18 + s) * plane + d.at(x, y0));
  char* opf = reinterpret_cast<char*>(Sout + 9 * s * plane + d.at(x, y0));                    // own species
  char* opg = reinterpret_cast<char*>(Sout + (18 + s) * plane + d.at(x, y0));                 // own thermal half
  const long long sofs = s ? 5 * planeB : 0;                                                     // planes 0.. -> 6.. for lane 1 (gp, opg carry + s)
  const int co = s ? kB : -kB;                                                                    // x - c_x of c_1 / c_3

  // thermal populations of (x, y).  Lane s = 0 reads
  // g_0, g_1, g_2, g_5, g_6 at x - c_i; lane s = 1 the opposite directions at x + c_i.
  double g0 = 0.0, ga = 0.0, gb = 0.0, gc = 0.0, gd = 0.0;
  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;  // MODE 3: s = 0 {mass_A, sum |u^(H)|^2, sum u_y^(H) T}; s = 1 {mass_B, sum d_y T, fluid sites}
  auto load_g = [&](int y) {
    long long rofs = s ? rowB : -rowB;  // row y - c_y of this lane's c_y = +-1 directions
    if (PERIODIC) {
      if (!s && y == 0) rofs = (long long)(ny - 1) * rowB;
      if (s && y == ny - 1) rofs = -(long long)(ny - 1) * rowB;
    }
    rofs += sofs;
    g0 = ldg_stream(reinterpret_cast<const ST*>(gp + 3 * planeB), pol);  // lane 1 reads g_1 here and never uses it
    ga = ldg_stream(reinterpret_cast<const ST*>(gp + 4 * planeB + co), pol);
    gb = ldg_stream(reinterpret_cast<const ST*>(gp + rofs), pol);
    gc = ldg_stream(reinterpret_cast<const ST*>(gp + 1 * planeB + rofs + co), pol);
    gd = ldg_stream(reinterpret_cast<const ST*>(gp + 2 * planeB + rofs - co), pol);
  };

  // L2 prefetch of the 9 thermal plane rows that phase 2 of row yp will load (one elected lane)
  auto prefetch_g = [&](int yp) {
    if (!(MODE == 1 || MODE == 3 || d.thermal) || yp >= y1) return;
    int ym = yp - 1, yq = yp + 1;
    if (PERIODIC) {
      if (ym < 0) ym = ny - 1;
      if (yq >= ny) yq = 0;
    }
    if (kTensor && (!PERIODIC || (yp > 0 && yp < ny - 1))) {
      tma_prefetch_4d(&tm.g, kXL + x0 - kHX, yp, 0, 0);
    } else {
      const long long o0 = d.at(x0 - kHX, yp), om = d.at(x0 - kHX, ym), op = d.at(x0 - kHX, yq);
#pragma unroll
      for (int i = 0; i < 9; i++) {
        const long long o = cy(i) == 0 ? o0 : (cy(i) > 0 ? om : op);
        prefetch_l2(Sin + (18 + pslot(i)) * plane + o, kCopyW * kB);
      }
    }
  };

  constexpr int kLag = TAU1 ? 3 : 2;  // rows between phase 1 and phase 2
  uint32_t parity = 0;  // one bit per slot
  for (int q = 0; q < q_end + (kLag - 2); q++) {
    const int r = y0 - 2 + q;
    const int slot = slot_of(q), rq = q % kRingRows;
    const bool p1 = q < q_end;  // phase 1 has a row (TAU1 runs one more iteration for the last phase 2)
    const bool valid = p1 && row_valid(r);
    const uint8_t s0 = m0, s1 = m1;
    if (q + 1 < q_end) {  // mask of the next row, a full iteration ahead of its use
      m0 = mask_at(r + 1, k);
      if (extra) m1 = mask_at(r + 1, kWC + k);
    }
    const int y = r - kLag;     // row of phase 2
    const bool do2 = y >= y0;
    if (do2 && (MODE == 1 || MODE == 3 || d.thermal)) load_g(y);  // consumed after the force stencil (a row earlier measured slower)
    // tau = 1: a landed row is dead when the iteration of its row ends (every warp arrives on the slot's "empty" barrier
    // there, after it has consumed what it loaded); the warps take turns re-arming: row q + 1 goes into the slot of row
    // q - 2, free for a whole iteration, so the wait below does not spin.  (Two rows ahead measured 8 % slower: the
    // issuer then waits for the slowest warp of the previous row.)
    if (TAU1 && wid == ((q - 1) & (kWarps - 1)) && lane == 0) {
      const int qi = q + 1;
      if (qi < q_end) {
        if (qi >= 3) mbar_wait(&sm.empty[slot_of(qi)], ((qi - 3) / 3) & 1u);
        issue(qi);
      }
      prefetch_g(y0 + q - 2 - kLag + kGPrefetchRows);  // phase 2 of that row runs kGPrefetchRows iterations from now
    }
    // ---- (1) rho_s, psi^s_s of row r (Eqs. (4), (12)); wall values at solid / out-of-domain nodes (L155, R9)
    if (valid) {
      mbar_wait(&sm.full[slot], (parity >> slot) & 1u);
      parity ^= 1u << slot;
    }
    if (TAU1) {
      // branch-free: every lane runs both passes (lanes >= 8 redo a halo column in the second and store nothing), solid
      // and out-of-domain nodes take the wall values by selection, so that phases 1 and 2 share one basic block
      if (p1) {
#pragma unroll
        for (int pass = 0; pass < 2; pass++) {
          const int c = pass == 0 ? k : kWC + (k & 3);
          const bool act = pass == 0 || extra;
          const uint8_t sol = pass == 0 ? s0 : s1;
          const ST* fs = &sm.f[slot][9 * s][kWC * wid + c + 2];  // S(x) of ring column c
          double f[9];
#pragma unroll
          for (int i = 0; i < 9; i++) f[i] = (double)fs[pslot(i) * kSW - cx(i)];
          const double rc = sum9(f);
          const double pc = d.rho0 * (1.0 - exp_nonpos(-rc * d.inv_rho0));
          const double rl = sol ? rho_wall : rc, pl = sol ? pss_wall : pc;
          if (act) {
            rho_r[rq][c][s] = rl;
            psi_r[rq][c][s] = pl;
            flag[rq][c] = sol;
            if (c >= 2 && c < kWC + 2)  // an interior column: its momentum, Eq. (5), for phase 2 three rows later
              sm.jr[wid][q & 3][c - 2][s] = make_double2(((f[1] - f[3]) + (f[5] - f[6])) + (f[8] - f[7]),
                                                         ((f[2] - f[4]) + (f[5] - f[7])) + (f[6] - f[8]));
          }
        }
      }
    } else {
#pragma unroll
    for (int pass = 0; pass < 2; pass++) {
      if (pass == 1 && !extra) break;
      const int c = pass == 0 ? k : kWC + k;
      const uint8_t sol = pass == 0 ? s0 : s1;
      double rl = rho_wall, pl = pss_wall;
      if (!sol) {
        const ST* fs = &sm.f[slot][9 * s][kWC * wid + c + 2];  // S(x) of ring column c
        double f[9];
#pragma unroll
        for (int i = 0; i < 9; i++) f[i] = (double)fs[pslot(i) * kSW - cx(i)];
        rl = sum9(f);
        pl = d.rho0 * (1.0 - exp_nonpos(-rl * d.inv_rho0));
      }
      rho_r[rq][c][s] = rl;
      psi_r[rq][c][s] = pl;
      flag[rq][c] = sol;
    }
    }
    // the 9 own-species populations of (x, y), landed two iterations ago
    const int slot2 = (q + 2) & 3;  // == (q - 2) & 3
    double f[9];
    if (!TAU1) {
      const ST* fs = &sm.f[slot2][9 * s][kWC * wid + k + kHX];
#pragma unroll
      for (int i = 0; i < 9; i++) f[i] = (double)fs[pslot(i) * kSW - cx(i)];
    }
    if (!TAU1) __syncwarp();  // ring row r of this warp is complete
    if (do2) {

    // ---- (2) collide row y = r - 2, whose stencil rows y-2..y+2 = r-4..r are resident
    const int rq0 = (q + kRingRows - kLag) % kRingRows;  // ring row of y
    const int cc = k + 2;                             // ring column of x
    const bool fluid = x < nx && !flag[rq0][cc];
    const double rl = rho_r[rq0][cc][s], rn = rho_r[rq0][cc][1 - s], pl = psi_r[rq0][cc][s];
    // force sums over the 5x5 neighbourhood: cross (w, other species' rho), self (G_a w + G_r p, own psi^s)
    // The stencils are antisymmetric (the term of -c is minus the term of +c), so opposite neighbours are
    // paired first: one subtraction serves both force components.
    double Xx = 0, Xy = 0, Sx = 0, Sy = 0, Sx2 = 0, Sy2 = 0;  // S = S + S2: two dependency chains per component
#pragma unroll
    for (int dy = 0; dy <= 2; dy++) {
      const int slp = (q + kRingRows - kLag + dy) % kRingRows, slm = (q + 2 * kRingRows - kLag - dy) % kRingRows;
#pragma unroll
      for (int dx = -2; dx <= 2; dx++) {
        if (dy == 0 && dx <= 0) continue;  // one representative of every pair {c, -c}
        const int c2 = dx * dx + dy * dy;
        const double kk = c2 == 1 ? k1 : c2 == 2 ? k2 : c2 == 4 ? k4 : c2 == 5 ? k5 : k8;      // |component| = 1
        const double kd = c2 == 4 ? k4d : c2 == 5 ? k5d : k8d;                                  // |component| = 2
        const double dpsi = psi_r[slp][cc + dx][s] - psi_r[slm][cc - dx][s];
        double& ax = (dy & 1) ? Sx2 : Sx;
        double& ay = (dx & 1) ? Sy2 : Sy;
        if (dx > 0) ax += (dx == 1 ? kk : kd) * dpsi;
        if (dx < 0) ax -= (dx == -1 ? kk : kd) * dpsi;
        if (dy > 0) ay += (dy == 1 ? kk : kd) * dpsi;
        if (c2 <= 2) {
          const double drho = rho_r[slp][cc + dx][1 - s] - rho_r[slm][cc - dx][1 - s];
          if (dx != 0) Xx += (w_c2(c2) * dx) * drho;
          if (dy != 0) Xy += (w_c2(c2) * dy) * drho;
        }
      }
    }
    Sx += Sx2;
    Sy += Sy2;
    double Fx = -gx * rl * Xx - pl * Sx, Fy = -gx * rl * Xy - pl * Sy;
    // moments, Eqs. (5), (17): partial sums of this lane + the other species' lane
    const double Tp = (s ? 0.0 : g0) + ga + gb + gc + gd;
    const double T = Tp + pair(Tp);
    double jxl, jyl;
    if (TAU1) {
      const double2 jl = sm.jr[wid][(q + 1) & 3][k][s];  // row y = r - 3: written three iterations ago
      jxl = jl.x;
      jyl = jl.y;
    } else {
      jxl = ((f[1] - f[3]) + (f[5] - f[6])) + (f[8] - f[7]);
      jyl = ((f[2] - f[4]) + (f[5] - f[7])) + (f[6] - f[8]);
      // The slot these nine values came from is handed back at the end of the iteration (the arrive below).  Pin that order
      // down instead of leaving it to where the compiler happens to put things: this statement needs all nine loads
      // complete (j depends on f_1..f_8), and volatile asm statements keep their program order, so no load of slot2 can
      // be scheduled behind the arrive -- also in the modes where the values only feed register accumulators.
      asm volatile("" ::"d"(f[0]), "d"(jxl), "d"(jyl));
    }
    const double jx = jxl + pair(jxl), jy = jyl + pair(jyl);
    // Eq. (22) buoyancy (R12) and the x-acceleration extension
    const double dT = d.thermal ? (T - d.T_ref) : 0.0;
    Fy += rl * d.alpha_g * dT;
    Fx += rl * d.body_ax;
    const double rho = rl + rn;
    const double inv = rcp_pos(rho), invl = d.tau * rcp_pos(rl);
    const double ux = jx * inv, uy = jy * inv;                      // Eq. (5)
    const double Ftx = Fx + pair(Fx), Fty = Fy + pair(Fy);
    const double uHx = (jx + 0.5 * Ftx) * inv, uHy = (jy + 0.5 * Fty) * inv;  // L139
    if (MODE == 1) {
      if (x < nx) {
        const size_t o = (size_t)y * nx + x;
        double* o1 = s ? oRB : oRA;
        double* o2 = s ? oUy : oUx;
        if (fluid) {
          if (o1) o1[o] = rl;
          if (o2) o2[o] = s ? uHy : uHx;
          if (!s && oT) oT[o] = T;
        } else {  // solid site: report the wall values
          if (o1) o1[o] = rho_wall;
          if (o2) o2[o] = 0.0;
          if (!s && oT) oT[o] = d.T_wall(y);
        }
      }
    } else if (MODE == 3) {
      // a10: mass_l (north_star), E (L248, R11), Nu (Eq. (24), R10).  R10's face differences telescope over every
      // fluid-fluid link, so sum_fluid d_y T = sum over fluid sites of [solid above] T_w(y + 1) - [solid below] T_w(y - 1).
      if (fluid) {
        const int rqp = (q + kRingRows - kLag + 1) % kRingRows, rqm = (q + kRingRows - kLag - 1) % kRingRows;  // ring rows of y + 1, y - 1
        int yu = y + 1, yd = y - 1;
        if (PERIODIC) { yu = yu >= ny ? 0 : yu; yd = yd < 0 ? ny - 1 : yd; }
        acc0 += rl;
        if (!s) {
          acc1 += uHx * uHx + uHy * uHy;
          acc2 += uHy * T;
        } else {
          acc1 += (flag[rqp][cc] ? d.T_wall(yu) : 0.0) - (flag[rqm][cc] ? d.T_wall(yd) : 0.0);
          acc2 += 1.0;
        }
      }
    } else {
      // kinetic part of P_xy (R21): momentum flux sum_i c_ix c_iy f_i of the populations arriving at (x, y) ...
      const double kpre = TAU1 ? 0.0 : (f[5] - f[6]) + (f[7] - f[8]);
      // own species: Eq. (6) shifted velocity, Eqs. (2), (3)
      {
        const double vx = ux + Fx * invl, vy = uy + Fy * invl;
        const double usq = 1.0 - 1.5 * (vx * vx + vy * vy);
        const double w0 = d.omega * (wq(0) * rl), w1 = d.omega * (wq(1) * rl), w5 = d.omega * (wq(5) * rl);
        if (TAU1 || om1 == 0.0) {  // uniform branch
          f[0] = relax_tau1(w0, 0.0, usq);
          f[1] = relax_tau1(w1, vx, usq);
          f[2] = relax_tau1(w1, vy, usq);
          f[3] = relax_tau1(w1, -vx, usq);
          f[4] = relax_tau1(w1, -vy, usq);
          f[5] = relax_tau1(w5, vx + vy, usq);
          f[6] = relax_tau1(w5, -vx + vy, usq);
          f[7] = relax_tau1(w5, -vx - vy, usq);
          f[8] = relax_tau1(w5, vx - vy, usq);
        } else {
          f[0] = relax(f[0], w0, 0.0, usq, om1);
          f[1] = relax(f[1], w1, vx, usq, om1);
          f[2] = relax(f[2], w1, vy, usq, om1);
          f[3] = relax(f[3], w1, -vx, usq, om1);
          f[4] = relax(f[4], w1, -vy, usq, om1);
          f[5] = relax(f[5], w5, vx + vy, usq, om1);
          f[6] = relax(f[6], w5, -vx + vy, usq, om1);
          f[7] = relax(f[7], w5, -vx - vy, usq, om1);
          f[8] = relax(f[8], w5, vx - vy, usq, om1);
        }
      }
      if (MODE == 2) {
        // ... averaged with that of the populations leaving it, plus the interaction part: for every coupling
        // F = -G psi(x) sum_c k(c) psi'(x + c) c the tensor (G / 2) psi(x) sum_c k(c) psi'(x + c) c_x c_y.  Terms
        // of c and -c have the same c_x c_y and are paired; only |c|^2 = 2, 5, 8 have c_x c_y != 0.
        const double kpost = (f[5] - f[6]) + (f[7] - f[8]);
        double Is = 0.0, Ix = 0.0;
#pragma unroll
        for (int dy = 1; dy <= 2; dy++) {
          const int slp = (q + kRingRows - kLag + dy) % kRingRows, slm = (q + 2 * kRingRows - kLag - dy) % kRingRows;
#pragma unroll
          for (int dx = -2; dx <= 2; dx++) {
            if (dx == 0) continue;
            const int c2 = dx * dx + dy * dy;
            const double kk = c2 == 2 ? k2 : c2 == 5 ? k5 : k8;
            Is += (kk * (dx * dy)) * (psi_r[slp][cc + dx][s] + psi_r[slm][cc - dx][s]);
            if (c2 == 2) Ix += (w_c2(2) * (dx * dy)) * (rho_r[slp][cc + dx][1 - s] + rho_r[slm][cc - dx][1 - s]);
          }
        }
        const double pl_xy = 0.5 * (kpre + kpost) + 0.5 * (pl * Is + gx * rl * Ix);
        const double pxy = pl_xy + pair(pl_xy);
        if (!s && x < nx) out.pxy[(size_t)y * nx + x] = fluid ? pxy : 0.0;
      }
      // own half of the thermal set: Eqs. (16), (18) with u^(H); directions sgn * {c_1, c_2, c_5, c_6}
      if (MODE == 0 && d.thermal) {
        const double vx = sgn * uHx, vy = sgn * uHy;
        const double usq = 1.0 - 1.5 * (uHx * uHx + uHy * uHy);
        const double w0 = d.omega_g * (wq(0) * T), w1 = d.omega_g * (wq(1) * T), w5 = d.omega_g * (wq(5) * T);
        if (om1g == 0.0) {  // uniform branch
          g0 = relax_tau1(w0, 0.0, usq);
          ga = relax_tau1(w1, vx, usq);
          gb = relax_tau1(w1, vy, usq);
          gc = relax_tau1(w5, vx + vy, usq);
          gd = relax_tau1(w5, -vx + vy, usq);
        } else {
          g0 = relax(g0, w0, 0.0, usq, om1g);
          ga = relax(ga, w1, vx, usq, om1g);
          gb = relax(gb, w1, vy, usq, om1g);
          gc = relax(gc, w5, vx + vy, usq, om1g);
          gd = relax(gd, w5, -vx + vy, usq, om1g);
        }
      }
      if (MODE == 0 && fluid) {
#pragma unroll
        for (int i = 0; i < 9; i++) stg_stream(reinterpret_cast<ST*>(opf + pslot(i) * planeB), f[i], pol);
        if (d.thermal) {
          if (!s) stg_stream(reinterpret_cast<ST*>(opg + 3 * planeB), g0, pol);
          stg_stream(reinterpret_cast<ST*>(opg + 4 * planeB), ga, pol);
          stg_stream(reinterpret_cast<ST*>(opg + sofs), gb, pol);
          stg_stream(reinterpret_cast<ST*>(opg + 1 * planeB + sofs), gc, pol);
          stg_stream(reinterpret_cast<ST*>(opg + 2 * planeB + sofs), gd, pol);
        }
        if (x < kGhost || x >= nx - kGhost) {  // periodic images of this column (ghost columns)
          for (int pass = 0; pass < 2; pass++)
            for (int xg = pass ? x - nx : x + nx; pass ? xg >= -kGhost : xg < nx + kGhost; xg += pass ? -nx : nx) {
              const long long e = (long long)(xg - x) * kB;
#pragma unroll
              for (int i = 0; i < 9; i++) *reinterpret_cast<ST*>(opf + pslot(i) * planeB + e) = (ST)f[i];
              if (d.thermal) {
                if (!s) *reinterpret_cast<ST*>(opg + 3 * planeB + e) = (ST)g0;
                *reinterpret_cast<ST*>(opg + 4 * planeB + e) = (ST)ga;
                *reinterpret_cast<ST*>(opg + sofs + e) = (ST)gb;
                *reinterpret_cast<ST*>(opg + 1 * planeB + sofs + e) = (ST)gc;
                *reinterpret_cast<ST*>(opg + 2 * planeB + sofs + e) = (ST)gd;
              }
            }
        }
      }
    }
    gp += rowB;
    opf += rowB;
    opg += rowB;
    }  // do2
    if (TAU1) {
      __syncwarp();  // ring row r of this warp is complete; this warp has read the slot of row r for the last time
      if (lane == 0 && p1) mbar_arrive(&sm.empty[slot]);
    } else if (q >= 2) {
      // General tau: the populations of row r - 2 were read from slot2 for the collision above; every warp hands the slot
      // back HERE, after the values have been consumed (see the asm next to j above).  The warp whose ticket shows that it
      // is the last of the kWarps re-arms the slot with row q + 2 at once: the copy has a whole iteration to land.  Before
      // it issues the copy it waits on "empty" like the tau = 1 issuer does -- the wait cannot block (all arrivals are
      // in), it is there for its acquire: the other warps' reads of the slot are ordered before the copy that overwrites it.
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&sm.empty[slot2]);
        if ((slot_ticket(&sm.ticket[slot2]) & (kWarps - 1)) == kWarps - 1) {
          mbar_wait(&sm.empty[slot2], ((q - 2) >> 2) & 1u);  // completion number (q - 2) / 4 of this slot's barrier
          if (q + 2 < q_end) issue(q + 2);
          prefetch_g(y0 + q - 3 + kGPrefetchRows);  // phase 2 of that row runs kGPrefetchRows iterations after the next one starts
        }
      }
    }
  }
  if (MODE == 3) {
    // warp-level reduction over the 16 lanes of each species (fixed butterfly), then the 8 warps in a fixed order
    __syncthreads();  // all warps are done with the rings; reuse the first ring as scratch
    double* scratch = &sm.rho[0][0][0][0];
#pragma unroll
    for (int o = 2; o < 32; o <<= 1) {
      acc0 += __shfl_xor_sync(0xffffffffu, acc0, o);
      acc1 += __shfl_xor_sync(0xffffffffu, acc1, o);
      acc2 += __shfl_xor_sync(0xffffffffu, acc2, o);
    }
    if (lane < 2) {
      scratch[(wid * 2 + lane) * 3 + 0] = acc0;
      scratch[(wid * 2 + lane) * 3 + 1] = acc1;
      scratch[(wid * 2 + lane) * 3 + 2] = acc2;
    }
    __syncthreads();
    if (t < 6) {
      double a = 0.0;
      for (int w = 0; w < kWarps; w++) a += scratch[(w * 2 + t / 3) * 3 + t % 3];
      // order {mass_A, mass_B, sum u^2, sum u_y T, sum d_y T, count}
      const int slot = t == 0 ? 0 : t == 1 ? 2 : t == 2 ? 3 : t == 3 ? 1 : t;
      out.partials[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 6 + slot] = a;
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
template <typename ST>
__global__ void __launch_bounds__(256)
boundary_kernel(const Dev d, ST* __restrict__ S, const int* __restrict__ sites, int n_sites) {
  const int nx = d.nx, ny = d.ny;
  const int n_lo = d.wall_lo ? nx : 0, n_ghost = n_lo + (d.wall_hi ? nx : 0);  // ghost rows exist beyond flat walls only
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int node = k >> 3, i = (k & 7) + 1;
  if (node >= n_ghost + n_sites) return;
  int sx, sy;  // lattice coordinates of the solid node, sy in -1..ny
  if (node < n_ghost) {
    sx = node < n_lo ? node : node - n_lo;
    sy = node < n_lo ? -1 : ny;
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
  const double Tw = d.T_wall(sy);
  const long long plane = d.plane;
  const long long os = d.at(sx, sy), ox = d.at(x, y);
  const int io = opp(i);
  const int pi = pslot(i), po = pslot(io);
  ST va = S[po * plane + ox], vb = S[(9 + po) * plane + ox];
  // R20: a moving flat wall (ghost row, not a post) hands the population back with the wall's momentum,
  // f_i = f*_opp(i) + 2 w_i rho_l (c_i . u_w) / c_s^2; rho_l(x) = sum_j S_l,j(x) (collision conserves it)
  const double uw = sy < 0 ? d.u_wall_bottom : (sy >= ny ? d.u_wall_top : 0.0);
  if (uw != 0.0 && cx(i) != 0) {
    double ra = 0.0, rb = 0.0;
#pragma unroll
    for (int j = 0; j < 9; j++) { ra += (double)S[j * plane + ox]; rb += (double)S[(9 + j) * plane + ox]; }
    va = (ST)((double)va + 6.0 * wq(i) * ra * (cx(i) * uw));
    vb = (ST)((double)vb + 6.0 * wq(i) * rb * (cx(i) * uw));
  }
  const ST vg = d.thermal ? (ST)(-(double)S[(18 + po) * plane + ox] + 2.0 * wq(i) * Tw) : (ST)0;
  for (int xg = sx; xg < nx + kGhost; xg += nx) {  // the node and its right-hand images
    S[pi * plane + os + (xg - sx)] = va;
    S[(9 + pi) * plane + os + (xg - sx)] = vb;
    if (d.thermal) S[(18 + pi) * plane + os + (xg - sx)] = vg;
  }
  for (int xg = sx - nx; xg >= -kGhost; xg -= nx) {
    S[pi * plane + os + (xg - sx)] = va;
    S[(9 + pi) * plane + os + (xg - sx)] = vb;
    if (d.thermal) S[(18 + pi) * plane + os + (xg - sx)] = vg;
  }
}

static dim3 strip_grid(const Dev& d, int seg_rows, int rows) {
  return dim3((d.nx + kW - 1) / kW, (rows + seg_rows - 1) / seg_rows);
}

template <typename ST>
static cudaError_t configure_for() {
  cudaError_t e = cudaSuccess;
  auto set = [&](auto* k, size_t bytes) {
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  };
  const size_t b = sizeof(Smem<ST, false>), b1 = sizeof(Smem<ST, true>);
  set(fused_kernel<0, false, ST, false>, b); set(fused_kernel<0, true, ST, false>, b);
  set(fused_kernel<0, false, ST, true>, b1); set(fused_kernel<0, true, ST, true>, b1);
  set(fused_kernel<1, false, ST, false>, b); set(fused_kernel<1, true, ST, false>, b);
  set(fused_kernel<2, false, ST, false>, b); set(fused_kernel<2, true, ST, false>, b);
  set(fused_kernel<3, false, ST, false>, b); set(fused_kernel<3, true, ST, false>, b);
  return e;
}

int configure_kernels() {
  cudaError_t e = configure_for<double>();
  if (e == cudaSuccess) e = configure_for<float>();
  return e == cudaSuccess ? 0 : (int)e;
}

// Rows per CTA segment.  strips x segments should fill whole waves of 2 CTAs per SM on 148 SMs.  Large lattices: as many
// waves (up to 8) as keep a segment at 48 rows or more -- many short CTAs balance the SMs better than few long ones and
// keep the rows in flight closer together, while each segment costs 4 warm-up rows and a pipeline fill (same-box
// measurements, profiles/r02_experiments.md block K: config 3 best with 1 wave of 57-row segments, config 4 with 4 waves
// of 56, config 5 with 8 waves of 114).  Lattices too small for that: the wave count (1..4) with the best ratio of useful
// to marched rows, never below kMinSegRows rows (they are bound by the latency of the serial march).
constexpr int kMinSegRows = 2;
constexpr int kGoodSegRows = 48;
int default_seg_rows(int nx, int ny) {
  const int strips = (nx + kW - 1) / kW, slots = kCtasPerSM * 148;
  for (int waves = 8; waves >= 1; waves--) {
    int segs = waves * slots / strips;
    if (segs < 1) segs = 1;
    const int seg = (ny + segs - 1) / segs;
    if (seg >= kGoodSegRows) return seg;
  }
  int best_seg = ny;
  double best = -1.0;
  for (int waves = 1; waves <= 4; waves++) {
    int segs = waves * slots / strips;
    if (segs < 1) segs = 1;
    int seg = (ny + segs - 1) / segs;
    if (seg < kMinSegRows) seg = ny < kMinSegRows ? ny : kMinSegRows;
    segs = (ny + seg - 1) / seg;
    const int ctas = strips * segs;
    const int w = (ctas + slots - 1) / slots;
    const double cost = (double)w * (seg + 4);  // rows marched by the busiest slot, incl. warm-up rows
    double score = (double)ny * strips / slots / cost;  // 1 = perfect
    if (w == 1) score *= 0.97;  // a single wave cannot rebalance CTAs that run slow
    if (score > best + 1e-9) { best = score; best_seg = seg; }
  }
  return best_seg;
}

int fused_grid_ctas(const Dev& d, int seg_rows, int rows) {
  const dim3 g = strip_grid(d, seg_rows, rows);
  return (int)(g.x * g.y);
}

template <int MODE, typename ST>
static void launch_mode(const Dev& d, const void* Sin, void* Sout, int seg_rows, int ya, int yb, const FusedOut& out,
                        const TMaps& tm, cudaStream_t st) {
  const ST* in = static_cast<const ST*>(Sin);
  ST* o = static_cast<ST*>(Sout);
  const dim3 g = strip_grid(d, seg_rows, yb - ya);
  if constexpr (MODE == 0) {
    if (d.omega == 1.0) {  // tau = 1 (Table A.3 and every BASELINE config): the populations are not needed by the collision
      const size_t sm1 = sizeof(Smem<ST, true>);
      if (d.periodic_y) fused_kernel<0, true, ST, true><<<g, kThreads, sm1, st>>>(d, in, o, seg_rows, ya, yb, out, tm);
      else fused_kernel<0, false, ST, true><<<g, kThreads, sm1, st>>>(d, in, o, seg_rows, ya, yb, out, tm);
      return;
    }
  }
  const size_t sm = sizeof(Smem<ST, false>);
  if (d.periodic_y) fused_kernel<MODE, true, ST, false><<<g, kThreads, sm, st>>>(d, in, o, seg_rows, ya, yb, out, tm);
  else fused_kernel<MODE, false, ST, false><<<g, kThreads, sm, st>>>(d, in, o, seg_rows, ya, yb, out, tm);
}

// Launch the fused kernel in `mode` on local rows [ya, yb); returns the number of launches (0 for an empty range).
int launch_fused(const Dev& d, int mode, const void* Sin, void* Sout, int seg_rows, int ya, int yb, const FusedOut& out,
                 const TMaps* maps, cudaStream_t st) {
  if (yb <= ya) return 0;
  static const TMaps none{};
  const TMaps& tm = maps ? *maps : none;  // every handle has maps (tlb_create fails without them)
  if (seg_rows > yb - ya) seg_rows = yb - ya;
  if (seg_rows < 1) seg_rows = 1;
  const bool f32 = d.prec == 32;
  switch (mode) {
    case 0: f32 ? launch_mode<0, float>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st) : launch_mode<0, double>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st); break;
    case 1: f32 ? launch_mode<1, float>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st) : launch_mode<1, double>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st); break;
    case 2: f32 ? launch_mode<2, float>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st) : launch_mode<2, double>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st); break;
    default: f32 ? launch_mode<3, float>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st) : launch_mode<3, double>(d, Sin, Sout, seg_rows, ya, yb, out, tm, st); break;
  }
  return 1;
}

int launch_boundary(const Dev& d, void* S, const int* sites, int n_sites, cudaStream_t st) {
  const long long n = 8ll * ((d.wall_lo ? d.nx : 0) + (d.wall_hi ? d.nx : 0) + n_sites);
  if (n == 0) return 0;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  if (d.prec == 32) boundary_kernel<float><<<blocks, 256, 0, st>>>(d, static_cast<float*>(S), sites, n_sites);
  else boundary_kernel<double><<<blocks, 256, 0, st>>>(d, static_cast<double*>(S), sites, n_sites);
  return 1;
}

}  // namespace tlb
