// tlb_analysis.cu -- droplet analysis, second stage (PAPER section 2.4, Eq. (25); readings R23-R26 of
// DESIGN.md): digital Voronoi colouring of the lattice by the nearest droplet centre, Delaunay links read off the
// vertices of the digital Voronoi cells, droplet matching and T1 events between two frames, droplet Nusselt number.
// All of it is integer / index work decided by fp64 comparisons; the distance is evaluated with explicitly rounded
// multiplies and adds (no FMA contraction) so that every decision is the one a plain fp64 evaluation takes.
#include "tlb_internal.cuh"

namespace tlb {

namespace {

constexpr int kBig = 0x7fffffff;

__device__ __forceinline__ double offset_to(int a, double c, int n, bool periodic) {
  double d = __dsub_rn((double)a, c);
  if (periodic) {
    const double half = 0.5 * (double)n;
    if (d > half) d = __dsub_rn(d, (double)n);
    else if (d < -half) d = __dadd_rn(d, (double)n);
  }
  return d;
}

__device__ __forceinline__ int nearest_site(double c, int n, bool periodic) {
  int r = (int)floor(c + 0.5);
  if (periodic) { r %= n; if (r < 0) r += n; }
  else { if (r < 0) r = 0; if (r >= n) r = n - 1; }
  return r;
}

// ---- R23: digital Voronoi tessellation.  The centres are binned into a uniform grid of cells at least `g` sites
// wide; a site searches the rings of cells around its own until no unvisited cell can hold a nearer centre.
__device__ __forceinline__ int cell_of(double c, double inv_w, int cells) {
  int i = (int)floor(c * inv_w);
  return i < 0 ? 0 : (i >= cells ? cells - 1 : i);
}

__global__ void vor_count_kernel(VorGrid G, const double* __restrict__ centres, int n, int* __restrict__ count) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int c = cell_of(centres[2 * k + 1], G.inv_wy, G.gy) * G.gx + cell_of(centres[2 * k], G.inv_wx, G.gx);
  atomicAdd(&count[c], 1);
}

// exclusive prefix sum of v[0..m) in place by one CTA (m is small: cells, or droplets); v[m] = total
__global__ void scan_kernel(int* __restrict__ v, int m) {
  __shared__ int part[1024];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < m; base += 1024) {
    const int i = base + threadIdx.x;
    const int a = i < m ? v[i] : 0;
    part[threadIdx.x] = a;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const int t = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
      __syncthreads();
      part[threadIdx.x] += t;
      __syncthreads();
    }
    if (i < m) v[i] = carry + part[threadIdx.x] - a;
    __syncthreads();
    if (threadIdx.x == 0) carry += part[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) v[m] = carry;
}

__global__ void vor_fill_kernel(VorGrid G, const double* __restrict__ centres, int n, const int* __restrict__ start,
                                int* __restrict__ cursor, int* __restrict__ members) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int c = cell_of(centres[2 * k + 1], G.inv_wy, G.gy) * G.gx + cell_of(centres[2 * k], G.inv_wx, G.gx);
  members[start[c] + atomicAdd(&cursor[c], 1)] = k;
}

__global__ void vor_colour_kernel(const Dev d, VorGrid G, const double* __restrict__ centres, const int* __restrict__ start,
                                  const int* __restrict__ members, int* __restrict__ colour) {
  const int nx = d.nx, ny = d.ny;
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)nx * ny) return;
  const int x = (int)(q % nx), y = (int)(q / nx);
  const bool per = d.periodic_y != 0;
  const int ix = cell_of((double)x, G.inv_wx, G.gx), iy = cell_of((double)y, G.inv_wy, G.gy);
  int best = -1;
  double bd = 0.0;
  const int rmax = G.gx > G.gy ? G.gx : G.gy;
  for (int R = 0; R <= rmax; R++) {
    for (int dyc = -R; dyc <= R; dyc++) {
      int cyi = iy + dyc;
      if (per) { cyi %= G.gy; if (cyi < 0) cyi += G.gy; }
      else if (cyi < 0 || cyi >= G.gy) continue;
      const int step = (dyc == -R || dyc == R) ? 1 : 2 * R;  // the ring of Chebyshev radius R
      for (int dxc = -R; dxc <= R; dxc += step) {
        int cxi = (ix + dxc) % G.gx;
        if (cxi < 0) cxi += G.gx;
        const int c = cyi * G.gx + cxi;
        for (int m = start[c]; m < start[c + 1]; m++) {
          const int k = members[m];
          const double dx = offset_to(x, centres[2 * k], nx, true), dy = offset_to(y, centres[2 * k + 1], ny, per);
          const double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
          if (best < 0 || d2 < bd || (d2 == bd && k < best)) { best = k; bd = d2; }  // ties: the smallest index
        }
      }
    }
    // every centre in a cell not visited yet is farther than R cell widths (less one site of rounding slack)
    const double reach = (double)R * G.wmin - 1.0;
    if (best >= 0 && reach > 0.0 && bd <= reach * reach) break;
  }
  colour[q] = best;
}

// ---- R24: Delaunay links from the 2 x 2 blocks that hold at least three colours (the wall colour -1 beyond flat walls)
__device__ __forceinline__ void adj_insert(int* __restrict__ adj, int a, int b, int* __restrict__ overflow) {
  int* row = adj + (size_t)a * kMaxDegree;
  for (int j = 0; j < kMaxDegree; j++) {
    const int old = atomicCAS(&row[j], -1, b);
    if (old == -1 || old == b) return;
  }
  atomicExch(overflow, 1);
}

__global__ void del_vertex_kernel(const Dev d, const int* __restrict__ colour, int* __restrict__ adj, int* __restrict__ overflow) {
  const int nx = d.nx, ny = d.ny;
  const bool per = d.periodic_y != 0;
  const int rows = per ? ny : ny + 1;
  const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (size_t)nx * rows) return;
  const int x = (int)(q % nx), y = (int)(q / nx) - (per ? 0 : 1);
  const int x1 = x + 1 == nx ? 0 : x + 1;
  int y1 = y + 1;
  if (per && y1 == ny) y1 = 0;
  int c[4];
  c[0] = y < 0 ? -1 : colour[(size_t)y * nx + x];
  c[1] = y < 0 ? -1 : colour[(size_t)y * nx + x1];
  c[2] = y1 >= ny ? -1 : colour[(size_t)y1 * nx + x];
  c[3] = y1 >= ny ? -1 : colour[(size_t)y1 * nx + x1];
  int distinct = 1 + (c[1] != c[0]) + (c[2] != c[0] && c[2] != c[1]) + (c[3] != c[0] && c[3] != c[1] && c[3] != c[2]);
  if (distinct < 3) return;
  // sides 0-1, 2-3, 0-2, 1-3, main diagonal 0-3, anti-diagonal 1-2 (dropped in a four-colour block)
  const int pa[6] = {0, 2, 0, 1, 0, 1}, pb[6] = {1, 3, 2, 3, 3, 2};
#pragma unroll
  for (int e = 0; e < 6; e++) {
    if (distinct == 4 && e == 5) continue;
    int a = c[pa[e]], b = c[pb[e]];
    if (a < 0 || b < 0 || a == b) continue;
    if (a > b) { const int t = a; a = b; b = t; }
    adj_insert(adj, a, b, overflow);
  }
}

// sort every row of the table (empty slots last) and count its entries
__global__ void adj_sort_kernel(int* __restrict__ adj, int n, int* __restrict__ deg) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int v[kMaxDegree];
  int* row = adj + (size_t)a * kMaxDegree;
  int m = 0;
#pragma unroll
  for (int j = 0; j < kMaxDegree; j++) { const int t = row[j]; v[j] = t < 0 ? kBig : t; m += t >= 0; }
  for (int i = 1; i < kMaxDegree; i++) {
    const int t = v[i];
    int j = i - 1;
    while (j >= 0 && v[j] > t) { v[j + 1] = v[j]; j--; }
    v[j + 1] = t;
  }
#pragma unroll
  for (int j = 0; j < kMaxDegree; j++) row[j] = v[j] == kBig ? -1 : v[j];
  deg[a] = m;
}

__global__ void del_write_kernel(const int* __restrict__ adj, const int* __restrict__ offs, int n, int max_links,
                                 const int* __restrict__ overflow, int* __restrict__ n_links, int* __restrict__ links) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a == 0) *n_links = *overflow ? -1 : offs[n];
  if (a >= n) return;
  const int* row = adj + (size_t)a * kMaxDegree;
  const int o = offs[a], m = offs[a + 1] - o;
  for (int j = 0; j < m; j++)
    if (o + j < max_links) { links[2 * (o + j)] = a; links[2 * (o + j) + 1] = row[j]; }
}

// ---- R25: matching and T1 events
__global__ void match_kernel(const Dev d, const int* __restrict__ colour_past, const double* __restrict__ centres, int n,
                             int* __restrict__ map) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  map[i] = colour_past[(size_t)nearest_site(centres[2 * i + 1], d.ny, d.periodic_y != 0) * d.nx + nearest_site(centres[2 * i], d.nx, true)];
}

// displacement of every present droplet from its past partner (minimum image), (0, 0) without one
__global__ void displacement_kernel(const Dev d, const double* __restrict__ past, const double* __restrict__ now,
                                    const int* __restrict__ map, int n, double* __restrict__ disp) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double dx = 0.0, dy = 0.0;
  const int m = map[i];
  if (m >= 0) {
    dx = __dsub_rn(now[2 * i], past[2 * m]);
    dy = __dsub_rn(now[2 * i + 1], past[2 * m + 1]);
    const double hx = 0.5 * (double)d.nx, hy = 0.5 * (double)d.ny;
    if (dx > hx) dx -= (double)d.nx; else if (dx < -hx) dx += (double)d.nx;
    if (d.periodic_y) { if (dy > hy) dy -= (double)d.ny; else if (dy < -hy) dy += (double)d.ny; }
  }
  disp[2 * i] = dx;
  disp[2 * i + 1] = dy;
}

// symmetric adjacency table of a link list; `map` (nullable) rewrites the ends, links with an end < 0, beyond n or
// with equal ends are dropped
__global__ void adj_build_kernel(const int* __restrict__ links, int n_links, const int* __restrict__ map, int n_map, int n,
                                 int* __restrict__ adj, int* __restrict__ overflow) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_links) return;
  int a = links[2 * k], b = links[2 * k + 1];
  if (map) {
    a = (a >= 0 && a < n_map) ? map[a] : -1;
    b = (b >= 0 && b < n_map) ? map[b] : -1;
  }
  if (a < 0 || b < 0 || a >= n || b >= n || a == b) return;
  adj_insert(adj, a, b, overflow);
  adj_insert(adj, b, a, overflow);
}

__device__ __forceinline__ bool adj_has(const int* __restrict__ adj, int a, int b) {
  const int* row = adj + (size_t)a * kMaxDegree;
  bool f = false;
#pragma unroll 4
  for (int j = 0; j < kMaxDegree; j++) f |= row[j] == b;
  return f;
}

// one thread per past link a-b that is gone: common past neighbours c < d of a and b with c-d new and the four sides kept
__global__ void t1_find_kernel(const int* __restrict__ past, int n_past, int n, const int* __restrict__ adjP,
                               const int* __restrict__ adjC, int cap, int* __restrict__ count, int* __restrict__ tmp) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_past) return;
  const int a = past[2 * k], b = past[2 * k + 1];
  if (a < 0 || b < 0 || a >= n || b >= n || a == b) return;
  if (adj_has(adjC, a, b)) return;
  const int* ra = adjP + (size_t)a * kMaxDegree;
  for (int i = 0; i < kMaxDegree; i++) {
    const int c = ra[i];
    if (c < 0 || c == b || !adj_has(adjP, b, c) || !adj_has(adjC, a, c) || !adj_has(adjC, b, c)) continue;
    for (int j = 0; j < kMaxDegree; j++) {
      const int e = ra[j];
      if (e <= c || e == b || !adj_has(adjP, b, e) || !adj_has(adjC, a, e) || !adj_has(adjC, b, e)) continue;
      if (!adj_has(adjC, c, e) || adj_has(adjP, c, e)) continue;
      const int slot = atomicAdd(count, 1);
      if (slot < cap) { tmp[4 * slot] = a < b ? a : b; tmp[4 * slot + 1] = a < b ? b : a; tmp[4 * slot + 2] = c; tmp[4 * slot + 3] = e; }
    }
  }
}

// lexicographic rank of every event among the (distinct) events found
__global__ void t1_rank_kernel(const int* __restrict__ tmp, const int* __restrict__ count, int cap, int max_events,
                               const int* __restrict__ overflow, int* __restrict__ n_events, int* __restrict__ events) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int m = *count < cap ? *count : cap;
  if (i == 0) *n_events = (*overflow || *count > cap) ? -1 : *count;
  if (i >= m) return;
  const int e0 = tmp[4 * i], e1 = tmp[4 * i + 1], e2 = tmp[4 * i + 2], e3 = tmp[4 * i + 3];
  int rank = 0;
  for (int j = 0; j < m; j++) {
    const int f0 = tmp[4 * j], f1 = tmp[4 * j + 1], f2 = tmp[4 * j + 2], f3 = tmp[4 * j + 3];
    const bool less = f0 != e0 ? f0 < e0 : (f1 != e1 ? f1 < e1 : (f2 != e2 ? f2 < e2 : f3 < e3));
    rank += less;
  }
  if (rank < max_events) { events[4 * rank] = e0; events[4 * rank + 1] = e1; events[4 * rank + 2] = e2; events[4 * rank + 3] = e3; }
}

// ---- R26: droplet Nusselt number, Eq. (25).  The fields are needed at one site per droplet only, so they are evaluated
// there directly from the pull-form buffer (Eqs. (4)-(12), (17), (22), L139 written out for one site) instead of
// sweeping the lattice: a few hundred loads per droplet.
__device__ __forceinline__ double w_of(int c2) { return c2 == 1 ? 1.0 / 9.0 : (c2 == 2 ? 1.0 / 36.0 : 0.0); }
__device__ __forceinline__ double p_of(int c2) {
  return c2 == 1 ? 4.0 / 63.0 : c2 == 2 ? 4.0 / 135.0 : c2 == 4 ? 1.0 / 180.0 : c2 == 5 ? 2.0 / 945.0 : c2 == 8 ? 1.0 / 15120.0 : 0.0;
}
__device__ __forceinline__ int wrapc(int a, int n) { return a < 0 ? a + n : (a >= n ? a - n : a); }

// is node (x, y) solid (a wall row beyond the lattice counts); x any column within 4 of the lattice, y any row
__device__ __forceinline__ bool solid_at(const Dev& d, int x, int& y) {
  if (d.periodic_y) y = wrapc(y, d.ny);
  else if (y < 0 || y >= d.ny) return true;
  return d.solid[(size_t)y * d.nx + wrapc(x, d.nx)] != 0;
}
// sum over i of S_set,i(n - c_i) at a fluid node n = (x, y) (y in range): a density (set 0, 1) or the temperature (set 2)
template <typename ST>
__device__ __forceinline__ double moment0(const Dev& d, const ST* __restrict__ S, int set, int x, int y) {
  double a = 0.0;
#pragma unroll
  for (int i = 0; i < 9; i++) {
    int sy = y - cy(i);
    if (d.periodic_y) sy = wrapc(sy, d.ny);
    a += (double)S[(9 * set + pslot(i)) * d.plane + d.at(x - cx(i), sy)];
  }
  return a;
}

template <typename ST>
__global__ void droplet_nusselt_kernel(const Dev d, const ST* __restrict__ S, const double* __restrict__ centres, int n,
                                       double tau_g, double* __restrict__ nu) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int nx = d.nx, ny = d.ny;
  const bool per = d.periodic_y != 0;
  const int x = nearest_site(centres[2 * i], nx, true), y = nearest_site(centres[2 * i + 1], ny, per);
  const double DT = d.T_bottom - d.T_top;
  if (d.solid[(size_t)y * nx + x] || DT == 0.0) { nu[i] = 0.0; return; }
  // moments of the site
  const double rA = moment0(d, S, 0, x, y), rB = moment0(d, S, 1, x, y), T = moment0(d, S, 2, x, y);
  double jy = 0.0;
#pragma unroll
  for (int k = 0; k < 9; k++) {
    if (cy(k) == 0) continue;
    int sy = y - cy(k);
    if (per) sy = wrapc(sy, ny);
    const long long o = d.at(x - cx(k), sy);
    jy += (double)cy(k) * ((double)S[pslot(k) * d.plane + o] + (double)S[(9 + pslot(k)) * d.plane + o]);
  }
  // y components of the interaction forces, Eqs. (7), (10), (11), wall values at solid nodes (L155)
  const double psA = d.rho0 * (1.0 - exp(-rA * d.inv_rho0)), psB = d.rho0 * (1.0 - exp(-rB * d.inv_rho0));
  double XA = 0.0, XB = 0.0, SA = 0.0, SB = 0.0;
  for (int dy = -2; dy <= 2; dy++)
    for (int dx = -2; dx <= 2; dx++) {
      const int c2 = dx * dx + dy * dy;
      if (c2 == 0 || dy == 0) continue;
      int yy = y + dy;
      double a, b, pa, pb;
      if (solid_at(d, x + dx, yy)) {
        a = d.rho_wall_A; b = d.rho_wall_B; pa = d.pss_wall_A; pb = d.pss_wall_B;
      } else {
        a = moment0(d, S, 0, x + dx, yy); b = moment0(d, S, 1, x + dx, yy);
        pa = d.rho0 * (1.0 - exp(-a * d.inv_rho0)); pb = d.rho0 * (1.0 - exp(-b * d.inv_rho0));
      }
      XA += w_of(c2) * dy * b;  // cross force on A sees psi^x of B, and the other way round
      XB += w_of(c2) * dy * a;
      SA += (d.G11a * w_of(c2) + d.G11r * p_of(c2)) * dy * pa;
      SB += (d.G22a * w_of(c2) + d.G22r * p_of(c2)) * dy * pb;
    }
  const double gx = d.G12 * d.inv_rho0 * d.inv_rho0;
  const double dTb = d.thermal ? (T - d.T_ref) : 0.0;
  const double FAy = -gx * rA * XA - psA * SA + rA * d.alpha_g * dTb;
  const double FBy = -gx * rB * XB - psB * SB + rB * d.alpha_g * dTb;
  const double uy = (jy + 0.5 * (FAy + FBy)) / (rA + rB);  // L139
  // d_y T as in Eq. (24) / R10
  int yu = y + 1, yd = y - 1;
  const bool su = solid_at(d, x, yu), sd = solid_at(d, x, yd);
  const double up = su ? d.T_wall(y + 1) : 0.5 * (T + moment0(d, S, 2, x, yu));
  const double dn = sd ? d.T_wall(y - 1) : 0.5 * (T + moment0(d, S, 2, x, yd));
  const double kappa = (tau_g - 0.5) / 3.0;
  nu[i] = (uy * T - kappa * (up - dn)) / (kappa * DT / ny);
}

unsigned blocks_of(long long n, int t) { return (unsigned)((n + t - 1) / t); }

}  // namespace

VorGrid make_vor_grid(int nx, int ny, int n) {
  VorGrid G;
  double g = n > 0 ? std::sqrt((double)nx * (double)ny / (double)n) : (double)nx;
  if (g < 8.0) g = 8.0;
  G.gx = (int)((double)nx / g); if (G.gx < 1) G.gx = 1;
  G.gy = (int)((double)ny / g); if (G.gy < 1) G.gy = 1;
  const double wx = (double)nx / G.gx, wy = (double)ny / G.gy;
  G.inv_wx = 1.0 / wx; G.inv_wy = 1.0 / wy;
  G.wmin = wx < wy ? wx : wy;
  return G;
}

// scratch: ints [cells + 1] start | [cells] cursor | [n] members
int launch_voronoi(const Dev& d, const double* centres, int n, int* scratch, int* colour, cudaStream_t st) {
  const size_t N = (size_t)d.nx * d.ny;
  if (n <= 0) { cudaMemsetAsync(colour, 0xff, N * sizeof(int), st); return 0; }
  const VorGrid G = make_vor_grid(d.nx, d.ny, n);
  const int cells = G.gx * G.gy;
  int* start = scratch;
  int* cursor = scratch + cells + 1;
  int* members = cursor + cells;
  cudaMemsetAsync(scratch, 0, (size_t)(2 * cells + 1) * sizeof(int), st);
  vor_count_kernel<<<blocks_of(n, 256), 256, 0, st>>>(G, centres, n, start);
  scan_kernel<<<1, 1024, 0, st>>>(start, cells);
  vor_fill_kernel<<<blocks_of(n, 256), 256, 0, st>>>(G, centres, n, start, cursor, members);
  vor_colour_kernel<<<blocks_of((long long)N, 256), 256, 0, st>>>(d, G, centres, start, members, colour);
  return 4;
}

// scratch: ints [n * kMaxDegree] adjacency | [n + 1] degrees / offsets | [1] overflow
int launch_delaunay(const Dev& d, const int* colour, int n, int* scratch, int max_links, int* n_links, int* links,
                    cudaStream_t st) {
  if (n <= 0) { cudaMemsetAsync(n_links, 0, sizeof(int), st); return 0; }
  int* adj = scratch;
  int* deg = adj + (size_t)n * kMaxDegree;
  int* overflow = deg + n + 1;
  cudaMemsetAsync(adj, 0xff, (size_t)n * kMaxDegree * sizeof(int), st);
  cudaMemsetAsync(deg, 0, (size_t)(n + 2) * sizeof(int), st);
  const long long blocks2 = (long long)d.nx * (d.periodic_y ? d.ny : d.ny + 1);
  del_vertex_kernel<<<blocks_of(blocks2, 256), 256, 0, st>>>(d, colour, adj, overflow);
  adj_sort_kernel<<<blocks_of(n, 128), 128, 0, st>>>(adj, n, deg);
  scan_kernel<<<1, 1024, 0, st>>>(deg, n);
  del_write_kernel<<<blocks_of(n, 256), 256, 0, st>>>(adj, deg, n, max_links, overflow, n_links, links);
  return 4;
}

int launch_displacements(const Dev& d, const double* past, const double* now, const int* map, int n, double* disp, cudaStream_t st) {
  if (n <= 0) return 0;
  displacement_kernel<<<blocks_of(n, 256), 256, 0, st>>>(d, past, now, map, n, disp);
  return 1;
}

int launch_match(const Dev& d, const int* colour_past, const double* centres_now, int n_now, int* map, cudaStream_t st) {
  if (n_now <= 0) return 0;
  match_kernel<<<blocks_of(n_now, 256), 256, 0, st>>>(d, colour_past, centres_now, n_now, map);
  return 1;
}

// scratch: ints [n * kMaxDegree] past table | [n * kMaxDegree] present table | [2] overflow, count | [4 * cap] events found
int launch_t1(const int* past, int n_past, const int* now, int n_now, const int* map, int n_map, int n, int* scratch, int cap,
              int max_events, int* n_events, int* events, cudaStream_t st) {
  if (n <= 0) { cudaMemsetAsync(n_events, 0, sizeof(int), st); return 0; }
  int* adjP = scratch;
  int* adjC = adjP + (size_t)n * kMaxDegree;
  int* overflow = adjC + (size_t)n * kMaxDegree;
  int* count = overflow + 1;
  int* tmp = count + 1;
  cudaMemsetAsync(adjP, 0xff, 2 * (size_t)n * kMaxDegree * sizeof(int), st);
  cudaMemsetAsync(overflow, 0, 2 * sizeof(int), st);
  int launches = 0;
  if (n_past > 0) { adj_build_kernel<<<blocks_of(n_past, 256), 256, 0, st>>>(past, n_past, nullptr, 0, n, adjP, overflow); launches++; }
  if (n_now > 0) { adj_build_kernel<<<blocks_of(n_now, 256), 256, 0, st>>>(now, n_now, map, n_map, n, adjC, overflow); launches++; }
  if (n_past > 0) { t1_find_kernel<<<blocks_of(n_past, 128), 128, 0, st>>>(past, n_past, n, adjP, adjC, cap, count, tmp); launches++; }
  t1_rank_kernel<<<blocks_of(cap > 0 ? cap : 1, 256), 256, 0, st>>>(tmp, count, cap, max_events, overflow, n_events, events);
  return launches + 1;
}

int launch_droplet_nusselt(const Dev& d, const void* S, const double* centres, int n, double tau_g, double* nu, cudaStream_t st) {
  if (n <= 0) return 0;
  if (d.prec == 32) droplet_nusselt_kernel<float><<<blocks_of(n, 64), 64, 0, st>>>(d, static_cast<const float*>(S), centres, n, tau_g, nu);
  else droplet_nusselt_kernel<double><<<blocks_of(n, 64), 64, 0, st>>>(d, static_cast<const double*>(S), centres, n, tau_g, nu);
  return 1;
}

}  // namespace tlb
