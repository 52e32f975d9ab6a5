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
    S[pslot(i) * d.plane + o] = (ST)va;
    S[(9 + pslot(i)) * d.plane + o] = (ST)vb;
    S[(18 + pslot(i)) * d.plane + o] = (ST)vc;
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
    if (a) a[i * n + q] = sol ? 0.0 : (double)S[pslot(i) * d.plane + o];
    if (b) b[i * n + q] = sol ? 0.0 : (double)S[(9 + pslot(i)) * d.plane + o];
    if (c) c[i * n + q] = sol ? 0.0 : (double)S[(18 + pslot(i)) * d.plane + o];
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

// ---- seeded input recipe (must reproduce inputs/__init__.py bit for bit) ----
__device__ __forceinline__ double uniform01(uint64_t seed, uint64_t stream, uint64_t k) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * ((stream << 40) + k + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  return __dmul_rn((double)(z >> 11), 1.0 / 9007199254740992.0);
}

// one CTA per droplet (centres in coordinates of the whole lattice): mark the sites of its disc in `inside`
__global__ void raster_kernel(const Dev d, const double* __restrict__ centres, double radius, uint8_t* __restrict__ inside) {
  const double cxd = centres[2 * blockIdx.x], cyd = centres[2 * blockIdx.x + 1];
  const int rr = (int)ceil(radius) + 1;
  const int bx = (int)floor(cxd) - rr, by = (int)floor(cyd) - rr, side = 2 * rr + 2;
  const double r2 = __dmul_rn(radius, radius);
  for (int t = threadIdx.x; t < side * side; t += blockDim.x) {
    const int y = by + t / side;  // row of the whole lattice (droplets never wrap in y)
    if (y < 0 || y >= d.ny_glob) continue;
    int x = (bx + t % side) % d.nx;
    if (x < 0) x += d.nx;
    double dx = fabs(__dsub_rn((double)x, cxd));
    dx = fmin(dx, __dsub_rn((double)d.nx, dx));
    const double dy = __dsub_rn((double)y, cyd);
    if (__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)) > r2) continue;
    // local images of that row: one, or none; a slab of a y-periodic lattice may hold it in a wrapped halo row
    for (int yl = y - d.y_off - (d.per_glob ? d.ny_glob : 0); yl < d.ny; yl += d.ny_glob)
      if (yl >= 0) inside[(size_t)yl * d.nx + x] = 1;
  }
}

__global__ void init_fields_kernel(const Dev d, const tlb_params p, uint64_t seed, const uint8_t* __restrict__ inside,
                                   uint8_t* __restrict__ solid, double* __restrict__ rhoA, double* __restrict__ rhoB,
                                   double* __restrict__ T) {
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)d.nx * d.ny) return;
  const int x = (int)(q % d.nx), y = d.gy((int)(q / d.nx));  // the recipe is stated on the whole lattice
  const uint64_t qg = (uint64_t)y * d.nx + x;
  bool sol = false;  // structured posts, reading R19
  if (p.post_w > 0 && p.post_h > 0 && p.post_period > 0)
    sol = (x % p.post_period) < p.post_w && (y < p.post_h || y >= d.ny_glob - p.post_h);
  solid[q] = sol ? 1 : 0;
  const bool in = inside[q] != 0;
  double a = in ? p.rho_in : p.rho_out, b = in ? p.rho_out : p.rho_in;
  if (!sol) {
    a = __dadd_rn(a, __dmul_rn(p.noise_amp, uniform01(seed, 1, qg)));
    b = __dadd_rn(b, __dmul_rn(p.noise_amp, uniform01(seed, 2, qg)));
  }
  rhoA[q] = a;
  rhoB[q] = b;
  const double yy = __dadd_rn((double)y, 0.5);  // linear profile between the walls, L314
  T[q] = __dadd_rn(__ddiv_rn(__dmul_rn(__dsub_rn(p.T_top, p.T_bottom), yy), (double)d.ny_glob), p.T_bottom);
}

// ---- observables (a10): the fused kernel (MODE 3) leaves per-CTA partial sums
// {mass_A, mass_B, sum |u^(H)|^2, sum u_y^(H) T, sum d_y T, fluid sites}; here they are combined in a fixed order ----
constexpr int kObsVals = 6;

// out4 = {mass_A, mass_B, E, Nu} from the six sums (whole lattice: after an all-reduce over slabs)
__device__ __forceinline__ void finish_observables(const Dev& d, const double* tot, double* out4) {
  const double nf = tot[5];
  const double kappa = (1.0 / d.omega_g - 0.5) / 3.0;  // Eq. (20)
  const double DT = d.T_bottom - d.T_top;
  out4[0] = tot[0];
  out4[1] = tot[1];
  out4[2] = nf > 0 ? tot[2] / nf : 0.0;                                                                      // L248, R11
  out4[3] = (nf > 0 && DT != 0.0) ? (tot[3] / nf - kappa * (tot[4] / nf)) / (kappa * DT / d.ny_glob) : 0.0;  // Eq. (24)
}

__global__ void observables_final_kernel(const Dev d, const double* __restrict__ partials, int n_blocks,
                                         double* __restrict__ sums6, double* __restrict__ out4) {
  __shared__ double tot[kObsVals];
  const int v = threadIdx.x >> 5, lane = threadIdx.x & 31;  // one warp per value, fixed lane order
  double a = 0.0;
  for (int b = lane; b < n_blocks; b += 32) a += partials[(size_t)b * kObsVals + v];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
  if (lane == 0) tot[v] = a;
  __syncthreads();
  if (threadIdx.x < kObsVals && sums6) sums6[threadIdx.x] = tot[threadIdx.x];
  if (threadIdx.x == 0 && out4) finish_observables(d, tot, out4);
}

__global__ void observables_from_sums_kernel(const Dev d, const double* __restrict__ sums6, double* __restrict__ out4) {
  double tot[kObsVals];
  for (int v = 0; v < kObsVals; v++) tot[v] = sums6[v];
  finish_observables(d, tot, out4);
}

// one CTA per row: x-average of a field plane over the fluid sites (u_av, Pxy_av of PAPER L248-250), fixed-order sums
__global__ void __launch_bounds__(256)
x_average_kernel(const Dev d, const double* __restrict__ ux, double* __restrict__ u_av) {
  const int y = blockIdx.x;
  if (y < d.own0 || y >= d.own1) {  // a slab's halo rows carry no fields
    if (threadIdx.x == 0) u_av[y] = 0.0;
    return;
  }
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

// ---- trapezoidal rough walls (reading R27): cut[j] = floor(j tan(alpha)) for the rows j = 0 .. height - 1 from the wall
__global__ void rough_walls_kernel(const Dev d, const int* __restrict__ cut, int height, int up, int down, int width,
                                   int lambda, int asymmetric, uint8_t* __restrict__ solid) {
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)d.nx * d.ny) return;
  const int x = (int)(q % d.nx), gy = d.gy((int)(q / d.nx));  // row of the whole lattice
  const int m = x % lambda;
  uint8_t v = 0;
  const int jd = gy, ju = d.ny_glob - 1 - gy;  // rows from the bottom / top wall
  if (down && jd < height) { const int r = cut[jd], l = asymmetric ? 0 : r; v |= (m >= l && m < width - r) ? 1 : 0; }
  if (up && ju < height) { const int r = cut[ju], l = asymmetric ? 0 : r; v |= (m >= l && m < width - r) ? 1 : 0; }
  solid[q] = v;
}

// ---- initial velocity perturbation (reading R29) on time-t populations in the ABI layout [9][ny][nx]
__global__ void perturb_kernel(const Dev d, double amplitude, double* __restrict__ fA, double* __restrict__ fB) {
  const size_t n = (size_t)d.nx * d.ny;
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n || d.solid[q]) return;
  const int x = (int)(q % d.nx), gy = d.gy((int)(q / d.nx));
  const double pi = 3.14159265358979323846;
  const double duy = amplitude * sin(2.0 * pi * (double)x / (double)d.nx) * sin(pi * ((double)gy + 0.5) / (double)d.ny_glob);
  double ra = 0.0, rb = 0.0;
#pragma unroll
  for (int i = 0; i < 9; i++) { ra += fA[i * n + q]; rb += fB[i * n + q]; }
#pragma unroll
  for (int i = 0; i < 9; i++) {
    const double cu = (double)cy(i) * duy;
    fA[i * n + q] += 3.0 * wq(i) * ra * cu;
    fB[i * n + q] += 3.0 * wq(i) * rb * cu;
  }
}

// ---- y-slab halo rows (tlb.h "Y-SLABS"): the kHalo owned rows next to a face <-> a contiguous buffer
// [27][kHalo][px] (whole padded rows, ghost columns included).  face 0 = low y, 1 = high y.
// pack reads the owned rows next to the face; unpack writes the halo rows beyond it.
template <bool UNPACK, typename ST>
__global__ void halo_copy_kernel(const Dev d, ST* __restrict__ S, int face, ST* __restrict__ buf) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= 27ll * kHalo * d.px) return;
  const int c = (int)(k % d.px), r = (int)((k / d.px) % kHalo), p = (int)(k / ((long long)d.px * kHalo));
  int y;
  if (UNPACK) y = face == 0 ? d.own0 - kHalo + r : d.own1 + r;
  else y = face == 0 ? d.own0 + r : d.own1 - kHalo + r;
  const long long o = p * d.plane + (long long)(y + 1) * d.row + c;
  if (UNPACK) S[o] = buf[k];
  else buf[k] = S[o];
}

// ---- droplet analysis, first stage (PAPER section 2.4, reading R22): bulk sites rho_A > B_th, clusters of
// nearest-neighbour (4-connected) bulk sites, x periodic (y too when the lattice is), label = smallest site index
// y nx + x of the cluster.  Lock-free union-find: every union hangs the larger root under the smaller one with
// atomicMin, so parents only decrease and the root of a finished cluster is its smallest index.
// One warp = 32 consecutive sites of one row.  A bulk site starts as a child of the leftmost site of its run of bulk
// sites inside the warp's window (a parent with a smaller index, like every parent later on): the horizontal bonds inside
// a window need no union at all.
__global__ void label_init_kernel(const Dev d, const double* __restrict__ rhoA, double threshold, int* __restrict__ labels) {
  const int x = blockIdx.y * blockDim.x + threadIdx.x, y = blockIdx.x;  // rows on grid.x (no 65535 limit)
  const size_t q = (size_t)y * d.nx + (x < d.nx ? x : 0);
  const bool bulk = x < d.nx && !d.solid[q] && rhoA[q] > threshold;
  const unsigned m = __ballot_sync(0xffffffffu, bulk);
  if (x >= d.nx) return;
  const int lane = threadIdx.x & 31;
  const unsigned holes_below = ~m & ((1u << lane) - 1u);           // non-bulk lanes to the left of this one
  const int start = holes_below ? 32 - __clz(holes_below) : 0;     // first lane of this lane's run
  labels[q] = bulk ? (int)q - (lane - start) : -1;
}

// rho_A = sum_i f_A,i (Eq. (4)) of the current state for the threshold: the 9 planes of the first fluid only, pulled
// from the pull-form buffer (ghost rows and columns hold what a fluid site pulls), same summation order as the fused kernel
template <typename ST>
__global__ void rho_a_kernel(const Dev d, const ST* __restrict__ S, double* __restrict__ rhoA) {
  const int x = blockIdx.y * blockDim.x + threadIdx.x, y = blockIdx.x;  // rows on grid.x (no 65535 limit)
  if (x >= d.nx) return;
  double f[9];
#pragma unroll
  for (int i = 0; i < 9; i++) {
    int sy = y - cy(i);
    if (d.periodic_y) sy = wrapi(sy, d.ny);
    f[i] = (double)S[pslot(i) * d.plane + d.at(x - cx(i), sy)];
  }
  rhoA[(size_t)y * d.nx + x] = (((f[0] + f[1]) + (f[2] + f[3])) + ((f[4] + f[5]) + (f[6] + f[7]))) + f[8];
}

__device__ __forceinline__ int find_root(volatile int* L, int i) {
  int cur = L[i];
  if (cur != i) {
    int prev = i, next;
    while (cur > (next = L[cur])) {  // path halving; a racing write can only store a smaller ancestor
      L[prev] = next;
      prev = cur;
      cur = next;
    }
  }
  return cur;
}

__device__ __forceinline__ void unite(int* L, int a, int b) {
  bool done;
  do {
    a = find_root(L, a);
    b = find_root(L, b);
    if (a < b) {
      const int old = atomicMin(&L[b], a);
      done = old == b;
      b = old;
    } else if (b < a) {
      const int old = atomicMin(&L[a], b);
      done = old == a;
      a = old;
    } else {
      done = true;
    }
  } while (!done);
}

// Bonds that still need a union: the horizontal bond into a warp window (its first lane and the site to its left, which
// for x = 0 is the periodic image x = nx - 1), and of the vertical bonds between two rows only the leftmost one of every
// stretch where both rows are bulk -- the bonds to its right connect the same two runs again.  (x = 0 never defers to
// its periodic left neighbour: two completely bulk rows would otherwise wait for one another all around the ring.)
__global__ void label_merge_kernel(const Dev d, int* __restrict__ labels) {
  const int x = blockIdx.y * blockDim.x + threadIdx.x, y = blockIdx.x;  // rows on grid.x (no 65535 limit)
  if (x >= d.nx) return;
  const size_t q = (size_t)y * d.nx + x;
  if (labels[q] < 0) return;
  const int xl = x > 0 ? x - 1 : d.nx - 1;
  const bool left = xl != x && labels[(size_t)y * d.nx + xl] >= 0;
  if (left && ((threadIdx.x & 31) == 0)) unite(labels, (int)q, y * d.nx + xl);  // x = 0 is lane 0 of its warp
  int yu = y + 1;
  if (yu >= d.ny) yu = d.periodic_y ? 0 : -1;
  if (yu >= 0 && yu != y && labels[(size_t)yu * d.nx + x] >= 0) {
    const bool left_pair = x > 0 && left && labels[(size_t)yu * d.nx + xl] >= 0;
    if (!left_pair) unite(labels, (int)q, yu * d.nx + x);
  }
}

// Every site takes the root of its tree.  Read-only chase (no path halving here: a halving store of a stale
// ancestor could land after, and undo, another thread's final write); concurrent final writes only ever replace a
// parent by the root of the same tree, so every chain stays valid while it is being read.
__global__ void label_flatten_kernel(const Dev d, int* __restrict__ labels) {
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)d.nx * d.ny) return;
  volatile int* L = labels;
  int cur = L[q];
  if (cur < 0) return;
  for (int next = L[cur]; next != cur; next = L[cur]) cur = next;
  L[q] = cur;
}

// roots (label == own index) appended in arrival order, then ranked: sorted[rank] = root
__global__ void droplet_roots_kernel(const Dev d, const int* __restrict__ labels, int* __restrict__ roots, int max_droplets,
                                     int* __restrict__ n_out) {
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)d.nx * d.ny) return;
  if (labels[q] != (int)q) return;
  const int k = atomicAdd(n_out, 1);
  if (k < max_droplets) roots[k] = (int)q;
}

__global__ void droplet_rank_kernel(const int* __restrict__ roots, int max_droplets, const int* __restrict__ n_out,
                                    int* __restrict__ sorted) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int n = min(*n_out, max_droplets);
  if (i >= n) return;
  const int r = roots[i];
  int rank = 0;
  for (int j = 0; j < n; j++) rank += roots[j] < r;
  sorted[rank] = r;
}

// signed minimum-image offset of a from b on a ring of n sites, in [-n/2, n/2)
__device__ __forceinline__ int min_image(int a, int b, int n) {
  int dlt = a - b;
  if (2 * dlt >= n) dlt -= n;
  else if (2 * dlt < -n) dlt += n;
  return dlt;
}

// per droplet: sites, sum of x offsets and of y offsets from the root site -- integer atomics, order-independent.
// The lanes of a warp (32 consecutive sites of a row) that belong to the same droplet add up first: one search and
// three atomics per group instead of per site.
__global__ void droplet_sums_kernel(const Dev d, const int* __restrict__ labels, const int* __restrict__ sorted,
                                    int max_droplets, const int* __restrict__ n_out, unsigned long long* __restrict__ sums) {
  const int x = blockIdx.y * blockDim.x + threadIdx.x, y = blockIdx.x;  // rows on grid.x (no 65535 limit)
  const int root = x < d.nx ? labels[(size_t)y * d.nx + x] : -1;
  const unsigned peers = __match_any_sync(0xffffffffu, root);
  int dx = 0, dy = 0;
  if (root >= 0) {
    const int xr = root % d.nx, yr = root / d.nx;
    dx = min_image(x, xr, d.nx);
    dy = d.periodic_y ? min_image(y, yr, d.ny) : y - yr;
  }
  const int sdx = __reduce_add_sync(peers, dx), sdy = __reduce_add_sync(peers, dy);
  if (root < 0 || (int)(threadIdx.x & 31) != __ffs(peers) - 1) return;  // the lowest lane of the group goes on
  const int n = min(*n_out, max_droplets);
  int lo = 0, hi = n;  // lower bound of root in sorted[0, n)
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (sorted[mid] < root) lo = mid + 1;
    else hi = mid;
  }
  if (lo >= n || sorted[lo] != root) return;  // a droplet beyond max_droplets
  atomicAdd(&sums[3 * lo + 0], (unsigned long long)__popc(peers));
  atomicAdd(&sums[3 * lo + 1], (unsigned long long)(long long)sdx);  // two's complement: wraps to the signed sum
  atomicAdd(&sums[3 * lo + 2], (unsigned long long)(long long)sdy);
}

// stats[k] = {label, sites, centre x, centre y} in ascending label order; centre = root + mean offset, wrapped
__global__ void droplet_finish_kernel(const Dev d, const int* __restrict__ sorted, const unsigned long long* __restrict__ sums,
                                      int max_droplets, const int* __restrict__ n_out, double* __restrict__ stats) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= min(*n_out, max_droplets)) return;
  const int root = sorted[k];
  const double cnt = (double)(long long)sums[3 * k];
  double cxm = (double)(root % d.nx) + __ddiv_rn((double)(long long)sums[3 * k + 1], cnt);
  double cym = (double)(root / d.nx) + __ddiv_rn((double)(long long)sums[3 * k + 2], cnt);
  if (cxm < 0.0) cxm += (double)d.nx;
  if (cxm >= (double)d.nx) cxm -= (double)d.nx;
  if (d.periodic_y) {
    if (cym < 0.0) cym += (double)d.ny;
    if (cym >= (double)d.ny) cym -= (double)d.ny;
  }
  stats[4 * k + 0] = (double)root;
  stats[4 * k + 1] = cnt;
  stats[4 * k + 2] = cxm;
  stats[4 * k + 3] = cym;
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
  build_links_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, sites, count);
  pad_mask_kernel<<<blocks_for((long long)d.px * d.ny, 256), 256, 0, st>>>(d, solidp);
  return 2;
}
int launch_init(const Dev& d, const tlb_params& p, uint64_t seed, const double* centres, int n_centres, uint8_t* inside,
                uint8_t* solid, double* rhoA, double* rhoB, double* T, cudaStream_t st) {
  int launches = 1;  // `inside` was zeroed by the caller
  if (n_centres > 0) {
    raster_kernel<<<n_centres, 128, 0, st>>>(d, centres, p.droplet_radius, inside);
    launches++;
  }
  init_fields_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, p, seed, inside, solid, rhoA, rhoB, T);
  return launches;
}
int launch_x_average(const Dev& d, const double* plane, double* av, cudaStream_t st) {
  x_average_kernel<<<d.ny, 256, 0, st>>>(d, plane, av);
  return 1;
}
int launch_observables_final(const Dev& d, const double* partials, int n_blocks, double* sums6, double* out4,
                             cudaStream_t st) {
  observables_final_kernel<<<1, 32 * kObsVals, 0, st>>>(d, partials, n_blocks, sums6, out4);
  return 1;
}
int launch_observables_from_sums(const Dev& d, const double* sums6, double* out4, cudaStream_t st) {
  observables_from_sums_kernel<<<1, 1, 0, st>>>(d, sums6, out4);
  return 1;
}
int launch_halo_pack(const Dev& d, const void* S, int face, void* buf, cudaStream_t st) {
  const long long n = 27ll * kHalo * d.px;
  if (d.prec == 32) halo_copy_kernel<false, float><<<blocks_for(n, 256), 256, 0, st>>>(d, const_cast<float*>(static_cast<const float*>(S)), face, static_cast<float*>(buf));
  else halo_copy_kernel<false, double><<<blocks_for(n, 256), 256, 0, st>>>(d, const_cast<double*>(static_cast<const double*>(S)), face, static_cast<double*>(buf));
  return 1;
}
int launch_halo_unpack(const Dev& d, void* S, int face, const void* buf, cudaStream_t st) {
  const long long n = 27ll * kHalo * d.px;
  if (d.prec == 32) halo_copy_kernel<true, float><<<blocks_for(n, 256), 256, 0, st>>>(d, static_cast<float*>(S), face, const_cast<float*>(static_cast<const float*>(buf)));
  else halo_copy_kernel<true, double><<<blocks_for(n, 256), 256, 0, st>>>(d, static_cast<double*>(S), face, const_cast<double*>(static_cast<const double*>(buf)));
  return 1;
}
int launch_rough_walls(const Dev& d, const int* cut, int height, int up, int down, int width, int lambda, int asymmetric,
                       uint8_t* solid, cudaStream_t st) {
  rough_walls_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, cut, height, up, down, width, lambda, asymmetric, solid);
  return 1;
}
int launch_perturb(const Dev& d, double amplitude, double* fA, double* fB, cudaStream_t st) {
  perturb_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, amplitude, fA, fB);
  return 1;
}
int launch_rho_a(const Dev& d, const void* S, double* rhoA, cudaStream_t st) {
  const dim3 g(d.ny, blocks_for(d.nx, 256));
  if (d.prec == 32) rho_a_kernel<float><<<g, 256, 0, st>>>(d, static_cast<const float*>(S), rhoA);
  else rho_a_kernel<double><<<g, 256, 0, st>>>(d, static_cast<const double*>(S), rhoA);
  return 1;
}
int launch_label_init(const Dev& d, const double* rhoA, double threshold, int* labels, cudaStream_t st) {
  label_init_kernel<<<dim3(d.ny, blocks_for(d.nx, 256)), 256, 0, st>>>(d, rhoA, threshold, labels);
  return 1;
}
int launch_label_merge(const Dev& d, int* labels, cudaStream_t st) {
  label_merge_kernel<<<dim3(d.ny, blocks_for(d.nx, 256)), 256, 0, st>>>(d, labels);
  return 1;
}
int launch_label_flatten(const Dev& d, int* labels, cudaStream_t st) {
  label_flatten_kernel<<<blocks_for((long long)d.nx * d.ny, 256), 256, 0, st>>>(d, labels);
  return 1;
}
// roots / sorted: [max_droplets] ints each, sums: [max_droplets][3] 64-bit (zeroed by the caller, like n_out);
// n_out: the number of droplets found; if it exceeds max_droplets the statistics are not meaningful
int launch_droplet_stats(const Dev& d, const int* labels, int* roots, int* sorted, unsigned long long* sums,
                         int max_droplets, int* n_out, double* stats, cudaStream_t st) {
  const unsigned nb = blocks_for((long long)d.nx * d.ny, 256);
  droplet_roots_kernel<<<nb, 256, 0, st>>>(d, labels, roots, max_droplets, n_out);
  droplet_rank_kernel<<<blocks_for(max_droplets, 256), 256, 0, st>>>(roots, max_droplets, n_out, sorted);
  droplet_sums_kernel<<<dim3(d.ny, blocks_for(d.nx, 256)), 256, 0, st>>>(d, labels, sorted, max_droplets, n_out, sums);
  droplet_finish_kernel<<<blocks_for(max_droplets, 256), 256, 0, st>>>(d, sorted, sums, max_droplets, n_out, stats);
  return 4;
}

}  // namespace tlb
