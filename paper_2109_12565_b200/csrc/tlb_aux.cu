// tlb_aux.cu -- state conversion (set / get populations and fields), boundary-link list, seeded
// initial state and the observable reductions (a10) of the CUDA path.
#include "tlb_internal.cuh"

namespace tlb {

namespace {

__device__ __forceinline__ int wrapi(int a, int n) { return a < 0 ? a + n : (a >= n ? a - n : a); }

// Is lattice node (x, y) (x already wrapped, y possibly out of range) a fluid site?
__device__ __forceinline__ bool fluid_at(const Dev& d, int x, int y) {
  if (d.periodic_y) y = wrapi(y, d.ny);
  else if (y < 0 || y >= d.ny) return false;
  return d.solid[(size_t)y * d.nx + x] == 0;
}

// One thread per node of the padded lattice (rows -1..ny, columns -kGhost..nx+kGhost-1; ghost columns
// are the periodic images).  S_i(s) = f_i(s + c_i) when s + c_i is a fluid site (Eq. (1) read
// backwards), else 0.  RHO = true: f_i = w_i * field (R14).
template <bool RHO, typename ST>
__global__ void scatter_kernel(const Dev d, const double* __restrict__ a, const double* __restrict__ b,
                               const double* __restrict__ c, ST* __restrict__ S) {
  const int nx = d.nx, ny = d.ny, wpad = nx + 2 * kGhost;
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= (long long)wpad * (ny + 2)) return;
  const int gx = (int)(k % wpad) - kGhost, sy = (int)(k / wpad) - 1;
  int sx = gx % nx;
  if (sx < 0) sx += nx;
  const size_t n = (size_t)nx * ny;
  const long long o = d.at(gx, sy);
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const int x = wrapi(sx + cx(i), nx);
    int y = sy + cy(i);
    double va = 0.0, vb = 0.0, vc = 0.0;
    const bool ghost_unused = d.periodic_y && (sy < 0 || sy >= ny);
    if (!ghost_unused && fluid_at(d, x, y)) {
      if (d.periodic_y) y = wrapi(y, ny);
      const size_t q = (size_t)y * nx + x;
      if (RHO) {
        va = wq(i) * a[q]; vb = wq(i) * b[q]; vc = wq(i) * c[q];
      } else {
        va = a[i * n + q]; vb = b[i * n + q]; vc = c[i * n + q];
      }
    }
    S[i * d.plane + o] = (ST)va;
    S[(9 + i) * d.plane + o] = (ST)vb;
    S[(18 + i) * d.plane + o] = (ST)vc;
  }
}

// f_i(x, t) = S_i(x - c_i); 0 on solid sites.
template <typename ST>
__global__ void gather_kernel(const Dev d, const ST* __restrict__ S, double* __restrict__ a,
                              double* __restrict__ b, double* __restrict__ c) {
  const int nx = d.nx, ny = d.ny;
  const size_t n = (size_t)nx * ny;
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n) return;
  const int x = (int)(q % nx), y = (int)(q / nx);
  const bool sol = d.solid[q] != 0;
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const int sx = wrapi(x - cx(i), nx);
    int sy = y - cy(i);
    if (d.periodic_y) sy = wrapi(sy, ny);
    const long long o = d.at(sx, sy);
    if (a) a[i * n + q] = sol ? 0.0 : (double)S[i * d.plane + o];
    if (b) b[i * n + q] = sol ? 0.0 : (double)S[(9 + i) * d.plane + o];
    if (c) c[i * n + q] = sol ? 0.0 : (double)S[(18 + i) * d.plane + o];
  }
}

template <typename ST>
__global__ void copy_g_kernel(const Dev d, const ST* __restrict__ src, ST* __restrict__ dst) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long per_row = 9ll * d.px;
  if (k >= per_row * (d.ny + 2)) return;
  const long long r = k / per_row, c = k % per_row;  // storage row, (thermal plane, column)
  const long long o = (18 + c / d.px) * d.plane + r * d.row + c % d.px;
  dst[o] = src[o];
}

// Solid in-domain sites with at least one fluid neighbour -> work list of the boundary kernel.
__global__ void build_links_kernel(const Dev d, int* __restrict__ sites, int* __restrict__ count) {
  const int nx = d.nx, ny = d.ny;
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)nx * ny) return;
  if (!d.solid[q]) return;
  const int x = (int)(q % nx), y = (int)(q / nx);
  bool touches = false;
#pragma unroll
  for (int i = 1; i < 9; i++) touches |= fluid_at(d, wrapi(x + cx(i), nx), y + cy(i));
  if (touches) sites[atomicAdd(count, 1)] = (int)q;
}

// Padded copy of the flag field for the fused kernel: [ny][px], lattice column x at kXL + x, ghost
// columns = periodic images, everything beyond them solid (never computed on).
__global__ void pad_mask_kernel(const Dev d, uint8_t* __restrict__ solidp) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= (size_t)d.px * d.ny) return;
  const int gx = (int)(k % d.px) - kXL, y = (int)(k / d.px);
  uint8_t v = 1;
  if (gx >= -kGhost && gx < d.nx + kGhost) {
    int x = gx % d.nx;
    if (x < 0) x += d.nx;
    v = d.solid[(size_t)y * d.nx + x] ? 1 : 0;
  }
  solidp[k] = v;
}

// ---- seeded input recipe (must reproduce paper_2109_12565_b200/inputs.py bit for bit) ----
__device__ __forceinline__ double uniform01(uint64_t seed, uint64_t stream, uint64_t k) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * ((stream << 40) + k + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  return __dmul_rn((double)(z >> 11), 1.0 / 9007199254740992.0);
}

// one CTA per droplet: mark the sites of its disc in `inside`
__global__ void raster_kernel(const Dev d, const double* __restrict__ centres, double radius, uint8_t* __restrict__ inside) {
  const double cxd = centres[2 * blockIdx.x], cyd = centres[2 * blockIdx.x + 1];
  const int rr = (int)ceil(radius) + 1;
  const int bx = (int)floor(cxd) - rr, by = (int)floor(cyd) - rr, side = 2 * rr + 2;
  const double r2 = __dmul_rn(radius, radius);
  for (int t = threadIdx.x; t < side * side; t += blockDim.x) {
    const int y = by + t / side;
    if (y < 0 || y >= d.ny) continue;
    int x = (bx + t % side) % d.nx;
    if (x < 0) x += d.nx;
    double dx = fabs(__dsub_rn((double)x, cxd));
    dx = fmin(dx, __dsub_rn((double)d.nx, dx));
    const double dy = __dsub_rn((double)y, cyd);
    if (__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)) <= r2) inside[(size_t)y * d.nx + x] = 1;
  }
}

__global__ void init_fields_kernel(const Dev d, const tlb_params p, uint64_t seed, const uint8_t* __restrict__ inside,
                                   uint8_t* __restrict__ solid, double* __restrict__ rhoA, double* __restrict__ rhoB,
                                   double* __restrict__ T) {
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)d.nx * d.ny) return;
  const int x = (int)(q % d.nx), y = (int)(q / d.nx);
  bool sol = false;  // structured posts, reading R19
  if (p.post_w > 0 && p.post_h > 0 && p.post_period > 0)
    sol = (x % p.post_period) < p.post_w && (y < p.post_h || y >= d.ny - p.post_h);
  solid[q] = sol ? 1 : 0;
  const bool in = inside[q] != 0;
  double a = in ? p.rho_in : p.rho_out, b = in ? p.rho_out : p.rho_in;
  if (!sol) {
    a = __dadd_rn(a, __dmul_rn(p.noise_amp, uniform01(seed, 1, q)));
    b = __dadd_rn(b, __dmul_rn(p.noise_amp, uniform01(seed, 2, q)));
  }
  rhoA[q] = a;
  rhoB[q] = b;
  const double yy = __dadd_rn((double)y, 0.5);  // linear profile between the walls, L314
  T[q] = __dadd_rn(__ddiv_rn(__dmul_rn(__dsub_rn(p.T_top, p.T_bottom), yy), (double)d.ny), p.T_bottom);
}

// ---- observables (a10): mass_A, mass_B, sum |u|^2, sum u_y T, sum d_y T, fluid count ----
constexpr int kObsThreads = 256;
constexpr int kObsVals = 6;

__device__ __forceinline__ double T_wall(const Dev& d, int y) { return (2 * y < d.ny) ? d.T_bottom : d.T_top; }

__global__ void __launch_bounds__(kObsThreads)
observables_partial_kernel(const Dev d, const double* __restrict__ rhoA, const double* __restrict__ rhoB,
                           const double* __restrict__ ux, const double* __restrict__ uy, const double* __restrict__ T,
                           double* __restrict__ partials) {
  const int nx = d.nx, ny = d.ny;
  const size_t n = (size_t)nx * ny;
  double acc[kObsVals] = {0, 0, 0, 0, 0, 0};
  for (size_t q = (size_t)blockIdx.x * kObsThreads + threadIdx.x; q < n; q += (size_t)gridDim.x * kObsThreads) {
    if (d.solid[q]) continue;
    const int x = (int)(q % nx), y = (int)(q / nx);
    const double t = T[q];
    acc[0] += rhoA[q];
    acc[1] += rhoB[q];
    acc[2] += ux[q] * ux[q] + uy[q] * uy[q];
    acc[3] += uy[q] * t;
    // R10: d_y T = Tface(y + 1/2) - Tface(y - 1/2); Tface = wall temperature at a solid neighbour
    int yu = y + 1, yd = y - 1;
    if (d.periodic_y) { yu = wrapi(yu, ny); yd = wrapi(yd, ny); }
    const double up = fluid_at(d, x, yu) ? 0.5 * (t + T[(size_t)yu * nx + x]) : T_wall(d, yu);
    const double dn = fluid_at(d, x, yd) ? 0.5 * (t + T[(size_t)yd * nx + x]) : T_wall(d, yd);
    acc[4] += up - dn;
    acc[5] += 1.0;
  }
  __shared__ double sh[kObsThreads / 32][kObsVals];
#pragma unroll
  for (int v = 0; v < kObsVals; v++) {
    double a = acc[v];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5][v] = a;
  }
  __syncthreads();
  if (threadIdx.x < kObsVals) {
    double a = 0.0;
    for (int w = 0; w < kObsThreads / 32; w++) a += sh[w][threadIdx.x];  // fixed order
    partials[(size_t)blockIdx.x * kObsVals + threadIdx.x] = a;
  }
}

__global__ void observables_final_kernel(const Dev d, const double* __restrict__ partials, int n_blocks,
                                         double* __restrict__ out4) {
  __shared__ double tot[kObsVals];
  const int v = threadIdx.x >> 5, lane = threadIdx.x & 31;  // one warp per value, fixed lane order
  double a = 0.0;
  for (int b = lane; b < n_blocks; b += 32) a += partials[(size_t)b * kObsVals + v];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
  if (lane == 0) tot[v] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    const double nf = tot[5];
    const double kappa = (1.0 / d.omega_g - 0.5) / 3.0;  // Eq. (20)
    const double DT = d.T_bottom - d.T_top;
    out4[0] = tot[0];
    out4[1] = tot[1];
    out4[2] = nf > 0 ? tot[2] / nf : 0.0;
    out4[3] = (nf > 0 && DT != 0.0) ? (tot[3] / nf - kappa * (tot[4] / nf)) / (kappa * DT / d.ny) : 0.0;  // Eq. (24)
  }
}

// one CTA per row: x-average of u_x over the fluid sites (u_av of PAPER L248-250), fixed-order sums
__global__ void __launch_bounds__(256)
x_average_kernel(const Dev d, const double* __restrict__ ux, double* __restrict__ u_av) {
  const int y = blockIdx.x;
  double a = 0.0, n = 0.0;
  for (int x = threadIdx.x; x < d.nx; x += 256)
    if (!d.solid[(size_t)y * d.nx + x]) { a += ux[(size_t)y * d.nx + x]; n += 1.0; }
  __shared__ double sa[8], sn[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); n += __shfl_down_sync(0xffffffffu, n, o); }
  if ((threadIdx.x & 31) == 0) { sa[threadIdx.x >> 5] = a; sn[threadIdx.x >> 5] = n; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double ta = 0.0, tn = 0.0;
    for (int w = 0; w < 8; w++) { ta += sa[w]; tn += sn[w]; }
    u_av[y] = tn > 0.0 ? ta / tn : 0.0;
  }
}

inline unsigned blocks_for(long long n, int t) { return (unsigned)((n + t - 1) / t); }

}  // namespace

int launch_scatter(const Dev& d, const double* fA, const double* fB, const double* g, void* S, cudaStream_t st) {
  const unsigned nb = blocks_for((long long)(d.nx + 2 * kGhost) * (d.ny + 2), 128);
  if (d.prec == 32) scatter_kernel<false, float><<<nb, 128, 0, st>>>(d, fA, fB, g, static_cast<float*>(S));
  else scatter_kernel<false, double><<<nb, 128, 0, st>>>(d, fA, fB, g, static_cast<double*>(S));
  return 1;
}
int launch_set_fields(const Dev& d, const double* rhoA, const double* rhoB, const double* T, void* S, cudaStream_t st) {
  const unsigned nb = blocks_for((long long)(d.nx + 2 * kGhost) * (d.ny + 2), 128);
  if (d.prec == 32) scatter_kernel<true, float><<<nb, 128, 0, st>>>(d, rhoA, rhoB, T, static_cast<float*>(S));
  else scatter_kernel<true, double><<<nb, 128, 0, st>>>(d, rhoA, rhoB, T, static_cast<double*>(S));
  return 1;
}
int launch_gather(const Dev& d, const void* S, double* fA, double* fB, double* g, cudaStream_t st) {
  const unsigned nb = blocks_for((long long)d.nx * d.ny, 128);
  if (d.prec == 32) gather_kernel<float><<<nb, 128, 0, st>>>(d, static_cast<const float*>(S), fA, fB, g);
  else gather_kernel<double><<<nb, 128, 0, st>>>(d, static_cast<const double*>(S), fA, fB, g);
  return 1;
}
int launch_copy_g(const Dev& d, const void* Ssrc, void* Sdst, cudaStream_t st) {
  const unsigned nb = blocks_for(9ll * d.px * (d.ny + 2), 256);
  if (d.prec == 32) copy_g_kernel<float><<<nb, 256, 0, st>>>(d, static_cast<const float*>(Ssrc), static_cast<float*>(Sdst));
  else copy_g_kernel<double><<<nb, 256, 0, st>>>(d, static_cast<const double*>(Ssrc), static_cast<double*>(Sdst));
  return 1;
}
int launch_build_links(const Dev& d, int* sites, int* count, uint8_t* solidp, cudaStream_t st) {
  cudaMemsetAsync(count, 0, sizeof(int), st);
  build_links_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, sites, count);
  pad_mask_kernel<<<blocks_for((long long)d.px * d.ny, 256), 256, 0, st>>>(d, solidp);
  return 2;
}
int launch_init(const Dev& d, const tlb_params& p, uint64_t seed, const double* centres, int n_centres, uint8_t* inside,
                uint8_t* solid, double* rhoA, double* rhoB, double* T, cudaStream_t st) {
  int launches = 1;
  cudaMemsetAsync(inside, 0, (size_t)d.nx * d.ny, st);
  if (n_centres > 0) {
    raster_kernel<<<n_centres, 128, 0, st>>>(d, centres, p.droplet_radius, inside);
    launches++;
  }
  init_fields_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, p, seed, inside, solid, rhoA, rhoB, T);
  return launches;
}
int launch_x_average(const Dev& d, const double* ux, double* u_av, cudaStream_t st) {
  x_average_kernel<<<d.ny, 256, 0, st>>>(d, ux, u_av);
  return 1;
}
int launch_observables(const Dev& d, const double* rhoA, const double* rhoB, const double* ux, const double* uy,
                       const double* T, double* partials, int n_blocks, double* out4, cudaStream_t st) {
  observables_partial_kernel<<<n_blocks, kObsThreads, 0, st>>>(d, rhoA, rhoB, ux, uy, T, partials);
  observables_final_kernel<<<1, 32 * kObsVals, 0, st>>>(d, partials, n_blocks, out4);
  return 2;
}

}  // namespace tlb
