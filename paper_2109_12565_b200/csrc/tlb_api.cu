// tlb_api.cu -- the C ABI of include/tlb.h: handle, parameter checks, workspace carving, and the
// host side of every call (argument marshalling and kernel launches only; no lattice arithmetic).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <new>
#include <vector>

#include "tlb_internal.cuh"

using namespace tlb;

struct tlb_handle {
  Dev d;
  tlb_params p;
  cudaStream_t st;
  int device;         // CUDA device of the workspace; every entry point runs with it current
  void* S[2];         // population buffers (pull form), 27 planes each, double or float (pop_precision)
  TMaps maps[2];      // tensor maps of S[0], S[1]
  bool has_maps;
  double* stage;      // [27][ny][nx] doubles for the *_host population calls when the buffers are float
  double* fld[5];     // rho_A, rho_B, u_x, u_y, T scratch planes
  uint8_t* solid;
  uint8_t* solidp;    // padded copy for the fused kernel
  int* sites;         // boundary work list
  int* count;
  double* partials;   // [obs_ctas][6] partial sums of the observables
  double* sums6;
  double* out4;
  int* n_drop;
  double* centres;
  int cur;            // S[cur] holds the current state
  int n_sites;
  int seg_rows;
  int obs_ctas;
  int halo_lo, halo_hi;  // y-slab: halo rows beyond the low / high face (0 at a wall or for a whole lattice)
  bool slab;
  bool step_open;     // between tlb_slab_step_edges and tlb_slab_step_finish
  bool has_state;
  cudaError_t err;
  int64_t launches;
  // CUDA graphs of kGraphSteps consecutive steps, one per starting buffer parity (launch-bound lattices)
  cudaStream_t cap_stream;
  cudaGraphExec_t gexec[2];
  int64_t g_launches[2];
  bool use_graph;
};

namespace {

size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

struct Geometry {  // local lattice of a handle
  int ny, y_off, own0, own1, halo_lo, halo_hi;
};

// Whole lattice: rows [0, ny_glob).  Slab: owned rows [y0, y1) plus kHalo imported rows beyond every face that is
// not a flat wall (a face of the whole lattice is one unless the lattice is periodic in y).
bool make_geometry(int ny_glob, int y0, int y1, bool slab, bool periodic, Geometry* g) {
  if (!slab) { *g = Geometry{ny_glob, 0, 0, ny_glob, 0, 0}; return true; }
  if (y0 < 0 || y1 > ny_glob || y1 <= y0) return false;
  g->halo_lo = (y0 == 0 && !periodic) ? 0 : kHalo;
  g->halo_hi = (y1 == ny_glob && !periodic) ? 0 : kHalo;
  if ((g->halo_lo || g->halo_hi) && y1 - y0 < kHalo) return false;  // a neighbour imports kHalo of these rows
  g->ny = (y1 - y0) + g->halo_lo + g->halo_hi;
  g->y_off = y0 - g->halo_lo;
  g->own0 = g->halo_lo;
  g->own1 = g->halo_lo + (y1 - y0);
  return true;
}

int obs_cta_count(int nx, int own_rows) {
  const int seg = default_seg_rows(nx, own_rows);
  return ((nx + kW - 1) / kW) * ((own_rows + seg - 1) / seg);
}

struct Layout {
  size_t S0, S1, stage, fld, solid, solidp, sites, count, partials, sums6, out4, n_drop, centres, total;
};

Layout make_layout(int nx, const Geometry& g, const tlb_params* p) {
  const int ny = g.ny;
  const size_t n = (size_t)nx * ny, px = (size_t)padded_pitch(nx), plane = px * (ny + 2);
  Layout L;
  size_t o = 0;
  const size_t esz = p->pop_precision == 32 ? sizeof(float) : sizeof(double);
  L.S0 = o; o = align_up(o + 27 * plane * esz);
  L.S1 = o; o = align_up(o + 27 * plane * esz);
  // fp64 buffers double as the staging area of the *_host population calls; fp32 buffers are too small
  L.stage = o; if (p->pop_precision == 32) o = align_up(o + 27 * n * sizeof(double));
  L.fld = o; o = align_up(o + 5 * n * sizeof(double));
  L.solid = o; o = align_up(o + n);
  L.solidp = o; o = align_up(o + px * ny);
  L.sites = o; o = align_up(o + n * sizeof(int));
  L.count = o; o = align_up(o + sizeof(int));
  L.partials = o; o = align_up(o + (size_t)obs_cta_count(nx, g.own1 - g.own0) * 6 * sizeof(double));
  L.sums6 = o; o = align_up(o + 6 * sizeof(double));
  L.out4 = o; o = align_up(o + 4 * sizeof(double));
  L.n_drop = o; o = align_up(o + sizeof(int));
  L.centres = o; o = align_up(o + 2 * sizeof(double) * (size_t)(p->n_droplets > 0 ? p->n_droplets : 1));
  L.total = o;
  return L;
}

bool params_ok(int nx, int ny, const tlb_params* p) {
  if (nx < 1 || ny < 1 || !p) return false;
  if ((long long)padded_pitch(nx) * (ny + 2 + 2 * kHalo) * 27 >= (1ll << 40)) return false;
  if ((long long)nx * (ny + 2 * kHalo) >= (1ll << 31)) return false;
  if (!(p->tau > 0.5) || !(p->tau_g > 0.5) || !(p->rho0 > 0.0)) return false;
  if (p->pop_precision != 64 && p->pop_precision != 32 && p->pop_precision != 0) return false;
  if (p->n_droplets < 0 || p->post_w < 0 || p->post_h < 0 || p->post_period < 0) return false;
  const bool posts = p->post_w > 0 && p->post_h > 0 && p->post_period > 0;
  if (posts && (p->periodic_y || 2 * p->post_h >= ny || p->post_w > p->post_period)) return false;
  if (p->periodic_y && (p->u_wall_bottom != 0.0 || p->u_wall_top != 0.0)) return false;  // no walls to move
  return true;
}

// Errors.  The handle keeps the first error of its OWN calls (sticky).  cudaGetLastError() is only read right
// after the handle's own launches (check()), and an error another library left pending on this thread is neither
// consumed nor adopted: enter() reports it without touching the handle.
int check(tlb_handle* h) {
  if (h->err == cudaSuccess) h->err = cudaGetLastError();
  return h->err == cudaSuccess ? TLB_OK : TLB_ECUDA;
}
int cu(tlb_handle* h, cudaError_t e) {
  if (h->err == cudaSuccess && e != cudaSuccess) h->err = e;
  return h->err == cudaSuccess ? TLB_OK : TLB_ECUDA;
}

// Makes the handle's device current for the duration of an entry point and restores the caller's.
struct Enter {
  int prev = -1, rc = TLB_OK;
  bool switched = false;
  explicit Enter(tlb_handle* h) {
    if (h->err != cudaSuccess) { rc = TLB_ECUDA; return; }
    if (cudaGetDevice(&prev) != cudaSuccess) { rc = TLB_ECUDA; return; }
    if (prev != h->device) {
      if (cudaSetDevice(h->device) != cudaSuccess) { rc = TLB_ECUDA; return; }
      switched = true;
    }
    if (cudaPeekAtLastError() != cudaSuccess) rc = TLB_ECUDA;  // somebody else's pending error: not ours to consume
  }
  ~Enter() { if (switched) cudaSetDevice(prev); }
};
#define TLB_ENTER(h)         \
  Enter enter_guard(h);      \
  if (enter_guard.rc != TLB_OK) return enter_guard.rc

constexpr int kGraphSteps = 16;

void drop_graphs(tlb_handle* h) {
  for (int k = 0; k < 2; k++)
    if (h->gexec[k]) { cudaGraphExecDestroy(h->gexec[k]); h->gexec[k] = nullptr; }
}

const TMaps* maps_of(const tlb_handle* h, const void* S) {
  return h->has_maps ? &h->maps[S == h->S[1] ? 1 : 0] : nullptr;
}

int launch_step(tlb_handle* h, const void* in, void* out, int ya, int yb, cudaStream_t st) {
  return launch_fused(h->d, 0, in, out, h->seg_rows, ya, yb, FusedOut{}, maps_of(h, in), st);
}

// Tensor maps of the two fp64 population buffers (layout: tlb_internal.cuh).  cuTensorMapEncodeTiled is a driver
// entry point; it is looked up at run time so that the library does not link against libcuda.
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool make_maps(tlb_handle* h) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  const encode_tiled_fn encode = reinterpret_cast<encode_tiled_fn>(fn);
  const Dev& d = h->d;
  const bool f32 = d.prec == 32;
  const cuuint64_t B = f32 ? sizeof(float) : sizeof(double);
  const CUtensorMapDataType dt = f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
  const cuuint64_t row = (cuuint64_t)d.row * B, plane = (cuuint64_t)d.plane * B;
  const cuuint64_t dims[5] = {(cuuint64_t)d.px, (cuuint64_t)d.ny + 2, 3, 3, 2};
  const cuuint64_t strides[4] = {row, plane, 3 * plane + row, 9 * plane};  // bytes, dimensions 1..4
  const cuuint32_t box[5] = {(cuuint32_t)(f32 ? kCopyW + 8 : kCopyW), 1, 3, 3, 2};  // = the slot row pitch of the fused kernel
  const cuuint32_t ones[5] = {1, 1, 1, 1, 1};
  for (int k = 0; k < 2; k++) {
    char* base = static_cast<char*>(h->S[k]);
    if (encode(&h->maps[k].f, dt, 5, base, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
    if (encode(&h->maps[k].g, dt, 4, base + 18 * plane, dims, strides, box, ones,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return false;
  }
  return true;
}

// Capture kGraphSteps steps starting from buffer parity `cur` (kernel arguments are baked in: the
// graph is dropped whenever the boundary work list changes).  Returns false if capture is not possible;
// the caller then launches the kernels one by one.
bool ensure_graph(tlb_handle* h, int cur) {
  if (h->gexec[cur]) return true;
  if (!h->use_graph || !h->cap_stream) return false;
  if (cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    h->use_graph = false;
    return false;
  }
  int64_t n = 0;
  int c = cur;
  for (int t = 0; t < kGraphSteps; t++) {
    n += launch_step(h, h->S[c], h->S[1 - c], h->d.own0, h->d.own1, h->cap_stream);
    n += launch_boundary(h->d, h->S[1 - c], h->sites, h->n_sites, h->cap_stream);
    c = 1 - c;
  }
  cudaGraph_t g = nullptr;
  cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
  if (e == cudaSuccess) e = cudaGraphInstantiate(&h->gexec[cur], g, 0);
  if (g) cudaGraphDestroy(g);
  if (e != cudaSuccess) {
    cudaGetLastError();
    h->gexec[cur] = nullptr;
    h->use_graph = false;
    return false;
  }
  h->g_launches[cur] = n;
  return true;
}

// After the mask changed: rebuild the boundary work list (count comes back to size the launch).
int rebuild_links(tlb_handle* h) {
  cu(h, cudaMemsetAsync(h->count, 0, sizeof(int), h->st));
  h->launches += launch_build_links(h->d, h->sites, h->count, h->solidp, h->st);
  int c = 0;
  cu(h, cudaMemcpyAsync(&c, h->count, sizeof(int), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  h->n_sites = c;
  drop_graphs(h);
  h->has_state = false;
  h->step_open = false;
  return check(h);
}

// The state in S[cur] was just written by a scatter: make the other buffer consistent (g planes are
// never rewritten when thermal = 0).
int after_state_set(tlb_handle* h) {
  if (!h->d.thermal) h->launches += launch_copy_g(h->d, h->S[h->cur], h->S[1 - h->cur], h->st);
  h->has_state = true;
  h->step_open = false;
  return check(h);
}

// SplitMix64-finaliser counter generator of the input recipe (host copy, for the droplet centres)
double uniform01_host(uint64_t seed, uint64_t stream, uint64_t k) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * ((stream << 40) + k + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z = z ^ (z >> 31);
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}

// Random sequential addition of equal discs, periodic in x.  Candidate k
// is accepted iff it keeps distance >= 2r + min_gap from every accepted centre; a cell list makes
// the test O(1).  Returns false if n discs could not be placed within 1000 n candidates.
bool place_droplets(int nx, int ny, uint64_t seed, const tlb_params& p, std::vector<double>& out) {
  const int n = p.n_droplets;
  out.clear();
  if (n == 0) return true;
  const double r = p.droplet_radius;
  const double y_lo = r + 3.0 + (double)p.post_h;
  const double y_hi = (double)ny - 1.0 - y_lo;
  if (y_hi < y_lo) return false;
  const double dmin = 2.0 * r + p.min_gap, dmin2 = dmin * dmin;
  const double cell = dmin > 1.0 ? dmin : 1.0;
  int gx = (int)std::floor((double)nx / cell), gy = (int)std::floor((double)ny / cell) + 1;
  if (gx < 1) gx = 1;
  const double cwx = (double)nx / gx;  // >= cell, so 3 cells cover dmin (all cells when gx < 3)
  std::vector<std::vector<int>> grid((size_t)gx * gy);
  const uint64_t kmax = 1000ull * (uint64_t)n;
  for (uint64_t k = 0; k < kmax && (int)(out.size() / 2) < n; k++) {
    const double cxd = uniform01_host(seed, 0, 2 * k) * (double)nx;
    const double t = uniform01_host(seed, 0, 2 * k + 1) * (y_hi - y_lo);
    const double cyd = y_lo + t;
    int ix = (int)(cxd / cwx), iy = (int)(cyd / cell);
    if (ix >= gx) ix = gx - 1;
    if (iy >= gy) iy = gy - 1;
    bool ok = true;
    for (int dj = -1; dj <= 1 && ok; dj++) {
      const int jy = iy + dj;
      if (jy < 0 || jy >= gy) continue;
      // x cells to look at: the three around ix (periodic), or the whole row when it has < 3 cells
      const int ncell = gx < 3 ? gx : 3;
      for (int t = 0; t < ncell && ok; t++) {
        const int c = gx < 3 ? t : ((ix - 1 + t) % gx + gx) % gx;
        for (int id : grid[(size_t)jy * gx + c]) {
          double dx = std::fabs(out[2 * id] - cxd);
          const double alt = (double)nx - dx;
          if (alt < dx) dx = alt;
          const double dy = out[2 * id + 1] - cyd;
          const double dd = dx * dx;
          const double ee = dy * dy;
          if (dd + ee < dmin2) { ok = false; break; }
        }
      }
    }
    if (!ok) continue;
    grid[(size_t)iy * gx + ix].push_back((int)(out.size() / 2));
    out.push_back(cxd);
    out.push_back(cyd);
  }
  return (int)(out.size() / 2) == n;
}

}  // namespace

extern "C" {

int tlb_default_params(tlb_params* p) {
  if (!p) return TLB_EINVAL;
  std::memset(p, 0, sizeof(*p));
  p->tau = 1.0; p->tau_g = 1.0; p->rho0 = 1.0;
  p->G12 = 0.405; p->G11a = -9.0; p->G11r = 8.1; p->G22a = -9.0; p->G22r = 8.1;
  p->rho_wall_A = 0.52; p->rho_wall_B = 0.52;
  p->T_bottom = 1.0; p->T_top = 0.0; p->T_ref = 0.5; p->alpha_g = 1e-4;
  p->droplet_radius = 6.0; p->min_gap = 4.0; p->rho_in = 1.0; p->rho_out = 0.04; p->noise_amp = 1e-3;
  p->thermal = 1; p->pop_precision = 64;
  return TLB_OK;
}

static int workspace_bytes_common(int nx, int ny_glob, int y0, int y1, bool slab, const tlb_params* p, size_t* bytes) {
  Geometry g;
  if (!bytes || !params_ok(nx, ny_glob, p) || !make_geometry(ny_glob, y0, y1, slab, p->periodic_y != 0, &g)) return TLB_EINVAL;
  *bytes = make_layout(nx, g, p).total;
  return TLB_OK;
}

int tlb_workspace_bytes(int nx, int ny, const tlb_params* p, size_t* bytes) {
  return workspace_bytes_common(nx, ny, 0, ny, false, p, bytes);
}

int tlb_slab_workspace_bytes(int nx, int ny, int y0, int y1, const tlb_params* p, size_t* bytes) {
  return workspace_bytes_common(nx, ny, y0, y1, true, p, bytes);
}

static int create_common(int nx, int ny_glob, int y0, int y1, bool slab, const tlb_params* p, void* workspace,
                         size_t workspace_bytes, void* stream, tlb_handle** out) {
  if (!out) return TLB_EINVAL;
  *out = nullptr;
  Geometry g;
  if (!params_ok(nx, ny_glob, p) || !workspace || ((uintptr_t)workspace & 255)) return TLB_EINVAL;
  if (!make_geometry(ny_glob, y0, y1, slab, p->periodic_y != 0, &g)) return TLB_EINVAL;
  const Layout L = make_layout(nx, g, p);
  if (workspace_bytes < L.total) return TLB_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return TLB_ECUDA;  // no CPU fallback
  }
  cudaPointerAttributes attr;
  if (cudaPointerGetAttributes(&attr, workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
    cudaGetLastError();
    return TLB_EINVAL;  // `workspace` is not device memory
  }
  tlb_handle* h = new (std::nothrow) tlb_handle();
  if (!h) return TLB_EINVAL;
  h->device = attr.device;
  h->err = cudaSuccess;
  Enter guard(h);
  if (guard.rc != TLB_OK) { delete h; return guard.rc; }
  const int ny = g.ny;
  char* w = static_cast<char*>(workspace);
  h->p = *p;
  h->st = static_cast<cudaStream_t>(stream);
  h->S[0] = w + L.S0;
  h->S[1] = w + L.S1;
  h->stage = p->pop_precision == 32 ? reinterpret_cast<double*>(w + L.stage) : nullptr;
  for (int k = 0; k < 5; k++) h->fld[k] = reinterpret_cast<double*>(w + L.fld) + (size_t)k * nx * ny;
  h->solid = reinterpret_cast<uint8_t*>(w + L.solid);
  h->solidp = reinterpret_cast<uint8_t*>(w + L.solidp);
  h->sites = reinterpret_cast<int*>(w + L.sites);
  h->count = reinterpret_cast<int*>(w + L.count);
  h->partials = reinterpret_cast<double*>(w + L.partials);
  h->sums6 = reinterpret_cast<double*>(w + L.sums6);
  h->out4 = reinterpret_cast<double*>(w + L.out4);
  h->n_drop = reinterpret_cast<int*>(w + L.n_drop);
  h->centres = reinterpret_cast<double*>(w + L.centres);
  h->slab = slab; h->halo_lo = g.halo_lo; h->halo_hi = g.halo_hi; h->step_open = false;
  Dev& d = h->d;
  d.nx = nx; d.ny = ny; d.thermal = p->thermal ? 1 : 0;
  d.y_off = g.y_off; d.ny_glob = ny_glob; d.per_glob = p->periodic_y ? 1 : 0;
  d.own0 = g.own0; d.own1 = g.own1;
  d.periodic_y = (!slab && p->periodic_y) ? 1 : 0;  // a slab is never periodic by itself: its faces import halo rows
  d.wall_lo = (!p->periodic_y && g.halo_lo == 0) ? 1 : 0;
  d.wall_hi = (!p->periodic_y && g.halo_hi == 0) ? 1 : 0;
  d.px = padded_pitch(nx);
  d.prec = p->pop_precision == 32 ? 32 : 64;
  // row-interleaved planes: the 27 plane rows of one lattice row lie next to one another ([ny + 2][27][px]), so the
  // rows a CTA works on sit in a few MB instead of being spread over 27 planes of the whole buffer (same-box A/B on
  // config 4 against plane-major [27][ny + 2][px]: 0.674 -> 0.652 ms)
  d.plane = d.px;
  d.row = 27ll * d.px;
  d.omega = 1.0 / p->tau; d.omega_g = 1.0 / p->tau_g; d.tau = p->tau;
  d.rho0 = p->rho0; d.inv_rho0 = 1.0 / p->rho0;
  d.G12 = p->G12; d.G11a = p->G11a; d.G11r = p->G11r; d.G22a = p->G22a; d.G22r = p->G22r;
  d.rho_wall_A = p->rho_wall_A; d.rho_wall_B = p->rho_wall_B;
  d.pss_wall_A = p->rho0 * (1.0 - std::exp(-p->rho_wall_A / p->rho0));  // Eq. (12) at the wall density
  d.pss_wall_B = p->rho0 * (1.0 - std::exp(-p->rho_wall_B / p->rho0));
  d.T_bottom = p->T_bottom; d.T_top = p->T_top; d.T_ref = p->T_ref; d.alpha_g = p->alpha_g; d.body_ax = p->body_ax;
  d.u_wall_bottom = p->u_wall_bottom; d.u_wall_top = p->u_wall_top;
  d.solid = h->solid;
  d.solidp = h->solidp;
  h->cur = 0; h->n_sites = 0; h->has_state = false; h->launches = 0;
  h->seg_rows = default_seg_rows(nx, g.own1 - g.own0);
  h->obs_ctas = obs_cta_count(nx, g.own1 - g.own0);
  h->gexec[0] = h->gexec[1] = nullptr;
  h->cap_stream = nullptr;
  h->use_graph = !(slab && (g.halo_lo || g.halo_hi));  // a slab's step is driven call by call (halo exchange in between)
  if (h->use_graph && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    h->cap_stream = nullptr;
    h->use_graph = false;
  }
  if (configure_kernels() != 0) { cudaGetLastError(); tlb_destroy(h); return TLB_ECUDA; }
  if (!make_maps(h)) { tlb_destroy(h); return TLB_ECUDA; }  // no second code path: fail loudly
  h->has_maps = true;
  cu(h, cudaMemsetAsync(h->solid, 0, (size_t)nx * ny, h->st));
  cu(h, cudaMemsetAsync(h->count, 0, sizeof(int), h->st));
  h->launches += launch_build_links(h->d, h->sites, h->count, h->solidp, h->st);  // padded mask of the empty flag field
  cu(h, cudaMemsetAsync(h->S[0], 0, 27 * (size_t)d.px * (ny + 2) * (d.prec == 32 ? sizeof(float) : sizeof(double)), h->st));
  cu(h, cudaMemsetAsync(h->S[1], 0, 27 * (size_t)d.px * (ny + 2) * (d.prec == 32 ? sizeof(float) : sizeof(double)), h->st));
  if (check(h) != TLB_OK) { tlb_destroy(h); return TLB_ECUDA; }
  *out = h;
  return TLB_OK;
}

int tlb_create(int nx, int ny, const tlb_params* p, void* workspace, size_t workspace_bytes, void* stream,
               tlb_handle** out) {
  return create_common(nx, ny, 0, ny, false, p, workspace, workspace_bytes, stream, out);
}

int tlb_create_slab(int nx, int ny, int y0, int y1, const tlb_params* p, void* workspace, size_t workspace_bytes,
                    void* stream, tlb_handle** out) {
  return create_common(nx, ny, y0, y1, true, p, workspace, workspace_bytes, stream, out);
}

int tlb_destroy(tlb_handle* h) {
  if (!h) return TLB_EINVAL;
  int prev = -1;
  cudaGetDevice(&prev);
  if (prev != h->device) cudaSetDevice(h->device);
  cudaStreamSynchronize(h->st);
  drop_graphs(h);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (prev >= 0 && prev != h->device) cudaSetDevice(prev);
  delete h;
  return TLB_OK;
}

int tlb_slab_layout(const tlb_handle* h, int32_t out6[6]) {
  if (!h || !out6) return TLB_EINVAL;
  out6[0] = h->d.ny; out6[1] = h->d.own0; out6[2] = h->d.own1; out6[3] = h->d.y_off; out6[4] = h->halo_lo; out6[5] = h->halo_hi;
  return TLB_OK;
}

int tlb_halo_bytes(const tlb_handle* h, size_t* bytes) {
  if (!h || !bytes) return TLB_EINVAL;
  *bytes = 27 * (size_t)kHalo * h->d.px * (h->d.prec == 32 ? sizeof(float) : sizeof(double));
  return TLB_OK;
}

int tlb_seg_rows(const tlb_handle* h) { return h ? h->seg_rows : TLB_EINVAL; }

// seeded initial state from a list of disc centres (host): posts from params, discs, noise, linear T (input recipe)
static int init_from_centres(tlb_handle* h, uint64_t seed, const std::vector<double>& c, double* dev_centres) {
  const int n = (int)(c.size() / 2);
  if (n > 0) {
    cu(h, cudaMemcpyAsync(dev_centres, c.data(), c.size() * sizeof(double), cudaMemcpyHostToDevice, h->st));
    cu(h, cudaStreamSynchronize(h->st));  // `c` is pageable and dies with the caller's frame
  }
  uint8_t* inside = reinterpret_cast<uint8_t*>(h->fld[2]);
  cu(h, cudaMemsetAsync(inside, 0, (size_t)h->d.nx * h->d.ny, h->st));
  h->launches += launch_init(h->d, h->p, seed, dev_centres, n, inside, h->solid, h->fld[0], h->fld[1], h->fld[4], h->st);
  int rc = rebuild_links(h);
  if (rc != TLB_OK) return rc;
  h->launches += launch_set_fields(h->d, h->fld[0], h->fld[1], h->fld[4], h->S[h->cur], h->st);
  return after_state_set(h);
}

int tlb_init(tlb_handle* h, uint64_t seed) {
  if (!h) return TLB_EINVAL;
  TLB_ENTER(h);
  std::vector<double> c;
  if (!place_droplets(h->d.nx, h->d.ny_glob, seed, h->p, c)) return TLB_EPLACEMENT;
  return init_from_centres(h, seed, c, h->centres);
}

int tlb_init_honeycomb(tlb_handle* h, int32_t ndx, int32_t ndy, uint64_t seed) {
  if (!h || ndx < 1 || ndy < 1) return TLB_EINVAL;
  const size_t N = (size_t)h->d.nx * h->d.ny;
  if (2 * (size_t)ndx * (size_t)ndy > N) return TLB_EINVAL;  // the centres are staged in a scratch plane
  TLB_ENTER(h);
  // inputs.honeycomb_centres, operation for operation (this file is compiled without FMA contraction)
  const double ax = (double)h->d.nx / (double)ndx;
  const double ay = ((double)h->d.ny_glob - 2.0 * (double)h->p.post_h) / (double)ndy;
  std::vector<double> c;
  c.reserve(2 * (size_t)ndx * ndy);
  for (int j = 0; j < ndy; j++)
    for (int i = 0; i < ndx; i++) {
      c.push_back(((double)i + 0.25 + 0.5 * (double)(j % 2)) * ax);
      c.push_back((double)h->p.post_h + ((double)j + 0.5) * ay);
    }
  return init_from_centres(h, seed, c, h->fld[3]);
}

int tlb_set_rough_walls(tlb_handle* h, const tlb_rough_walls* r) {
  if (!h || !r) return TLB_EINVAL;
  if (h->p.periodic_y || r->lambda < 1 || r->width < 0 || r->width > r->lambda || r->height < 0) return TLB_EINVAL;
  if ((r->up && r->down ? 2 * (long long)r->height : (long long)r->height) > h->d.ny_glob) return TLB_EINVAL;
  TLB_ENTER(h);
  std::vector<int> cut((size_t)(r->height > 0 ? r->height : 1), 0);
  const double t = std::tan(r->alpha);
  for (int j = 0; j < r->height; j++) cut[(size_t)j] = (int)std::floor((double)j * t);
  int* dcut = reinterpret_cast<int*>(h->fld[2]);  // height <= ny ints
  cu(h, cudaMemcpyAsync(dcut, cut.data(), cut.size() * sizeof(int), cudaMemcpyHostToDevice, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  h->launches += launch_rough_walls(h->d, dcut, r->height, r->up ? 1 : 0, r->down ? 1 : 0, r->width, r->lambda,
                                    r->asymmetric ? 1 : 0, h->solid, h->st);
  return rebuild_links(h);
}

int tlb_set_solid(tlb_handle* h, const uint8_t* solid) {
  if (!h || !solid) return TLB_EINVAL;
  TLB_ENTER(h);
  cu(h, cudaMemcpyAsync(h->solid, solid, (size_t)h->d.nx * h->d.ny, cudaMemcpyDeviceToDevice, h->st));
  return rebuild_links(h);
}

int tlb_set_solid_host(tlb_handle* h, const uint8_t* solid) {
  if (!h || !solid) return TLB_EINVAL;
  TLB_ENTER(h);
  cu(h, cudaMemcpyAsync(h->solid, solid, (size_t)h->d.nx * h->d.ny, cudaMemcpyHostToDevice, h->st));
  return rebuild_links(h);
}

int tlb_set_fields(tlb_handle* h, const double* rho_A, const double* rho_B, const double* T) {
  if (!h || !rho_A || !rho_B || !T) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_set_fields(h->d, rho_A, rho_B, T, h->S[h->cur], h->st);
  return after_state_set(h);
}

int tlb_set_fields_host(tlb_handle* h, const double* rho_A, const double* rho_B, const double* T) {
  if (!h || !rho_A || !rho_B || !T) return TLB_EINVAL;
  TLB_ENTER(h);
  const size_t b = (size_t)h->d.nx * h->d.ny * sizeof(double);
  cu(h, cudaMemcpyAsync(h->fld[0], rho_A, b, cudaMemcpyHostToDevice, h->st));
  cu(h, cudaMemcpyAsync(h->fld[1], rho_B, b, cudaMemcpyHostToDevice, h->st));
  cu(h, cudaMemcpyAsync(h->fld[4], T, b, cudaMemcpyHostToDevice, h->st));
  h->launches += launch_set_fields(h->d, h->fld[0], h->fld[1], h->fld[4], h->S[h->cur], h->st);
  int rc = after_state_set(h);
  cu(h, cudaStreamSynchronize(h->st));
  return rc != TLB_OK ? rc : check(h);
}

int tlb_set_populations(tlb_handle* h, const double* fA, const double* fB, const double* g) {
  if (!h || !fA || !fB || !g) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_scatter(h->d, fA, fB, g, h->S[h->cur], h->st);
  return after_state_set(h);
}

int tlb_get_populations(tlb_handle* h, double* fA, double* fB, double* g) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_gather(h->d, h->S[h->cur], fA, fB, g, h->st);
  return check(h);
}

// Host variants stage [27][ny][nx] through the buffer that is not current (it is rewritten by the
// next step anyway; its g planes are restored when thermal = 0).
int tlb_set_populations_host(tlb_handle* h, const double* fA, const double* fB, const double* g) {
  if (!h || !fA || !fB || !g) return TLB_EINVAL;
  TLB_ENTER(h);
  const size_t n9 = 9 * (size_t)h->d.nx * h->d.ny;
  double* stage = h->stage ? h->stage : static_cast<double*>(h->S[1 - h->cur]);
  cu(h, cudaMemcpyAsync(stage, fA, n9 * sizeof(double), cudaMemcpyHostToDevice, h->st));
  cu(h, cudaMemcpyAsync(stage + n9, fB, n9 * sizeof(double), cudaMemcpyHostToDevice, h->st));
  cu(h, cudaMemcpyAsync(stage + 2 * n9, g, n9 * sizeof(double), cudaMemcpyHostToDevice, h->st));
  h->launches += launch_scatter(h->d, stage, stage + n9, stage + 2 * n9, h->S[h->cur], h->st);
  // the staging area overlapped ghost / solid entries of the other buffer: they are dead until the
  // next boundary kernel rewrites them
  int rc = after_state_set(h);
  cu(h, cudaStreamSynchronize(h->st));
  return rc != TLB_OK ? rc : check(h);
}

int tlb_get_populations_host(tlb_handle* h, double* fA, double* fB, double* g) {
  if (!h || !fA || !fB || !g) return TLB_EINVAL;
  // while a slab step is open the other buffer holds the rows just computed and the halo rows being received:
  // staging through it would corrupt the step
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  const size_t n9 = 9 * (size_t)h->d.nx * h->d.ny;
  double* stage = h->stage ? h->stage : static_cast<double*>(h->S[1 - h->cur]);
  h->launches += launch_gather(h->d, h->S[h->cur], stage, stage + n9, stage + 2 * n9, h->st);
  cu(h, cudaMemcpyAsync(fA, stage, n9 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaMemcpyAsync(fB, stage + n9, n9 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaMemcpyAsync(g, stage + 2 * n9, n9 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  if (!h->d.thermal && !h->stage) h->launches += launch_copy_g(h->d, h->S[h->cur], h->S[1 - h->cur], h->st);
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

int tlb_perturb_velocity(tlb_handle* h, double amplitude) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  // time-t populations into the staging area, perturbed there, and back (the route of the *_host population calls)
  const size_t n9 = 9 * (size_t)h->d.nx * h->d.ny;
  double* stage = h->stage ? h->stage : static_cast<double*>(h->S[1 - h->cur]);
  h->launches += launch_gather(h->d, h->S[h->cur], stage, stage + n9, stage + 2 * n9, h->st);
  h->launches += launch_perturb(h->d, amplitude, stage, stage + n9, h->st);
  h->launches += launch_scatter(h->d, stage, stage + n9, stage + 2 * n9, h->S[h->cur], h->st);
  return after_state_set(h);
}

static std::string checkpoint_name(const char* dir, const char* stem, int index) {
  return std::string(dir) + "/" + stem + "_" + std::to_string(index) + ".in";
}

int tlb_write_checkpoint(tlb_handle* h, const char* dir, int32_t index) {
  if (!h || !dir) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  const size_t n9 = 9 * (size_t)h->d.nx * h->d.ny;
  std::vector<double> buf;
  try { buf.resize(3 * n9); } catch (...) { return TLB_EINVAL; }
  int rc = tlb_get_populations_host(h, buf.data(), buf.data() + n9, buf.data() + 2 * n9);
  if (rc != TLB_OK) return rc;
  const char* stems[3] = {"conf1", "conf2", "confG"};
  for (int k = 0; k < 3; k++) {
    FILE* f = std::fopen(checkpoint_name(dir, stems[k], index).c_str(), "wb");
    if (!f) return TLB_EIO;
    const size_t w = std::fwrite(buf.data() + k * n9, sizeof(double), n9, f);
    if (std::fclose(f) != 0 || w != n9) return TLB_EIO;
  }
  return TLB_OK;
}

int tlb_read_checkpoint(tlb_handle* h, const char* dir, int32_t index) {
  if (!h || !dir) return TLB_EINVAL;
  const size_t n9 = 9 * (size_t)h->d.nx * h->d.ny;
  std::vector<double> buf;
  try { buf.resize(3 * n9); } catch (...) { return TLB_EINVAL; }
  const char* stems[3] = {"conf1", "conf2", "confG"};
  for (int k = 0; k < 3; k++) {
    FILE* f = std::fopen(checkpoint_name(dir, stems[k], index).c_str(), "rb");
    if (!f) return TLB_EIO;
    const size_t r = std::fread(buf.data() + k * n9, sizeof(double), n9, f);
    const bool more = std::fgetc(f) != EOF;  // a dump of another lattice size
    std::fclose(f);
    if (r != n9 || more) return TLB_EIO;
  }
  return tlb_set_populations_host(h, buf.data(), buf.data() + n9, buf.data() + 2 * n9);
}

// ---- field files (Tables C.9, C.10; reading R31): plain host I/O after a read-back ----
static bool write_dat(const std::string& path, int nx, int ny, const double* a, const double* b) {
  FILE* f = std::fopen(path.c_str(), "w");
  if (!f) return false;
  bool ok = true;
  for (int y = 0; y < ny && ok; y++) {
    for (int x = 0; x < nx; x++) {
      const size_t q = (size_t)y * nx + x;
      const int r = b ? std::fprintf(f, "%d %d %.17g %.17g\n", x, y, a[q], b[q]) : std::fprintf(f, "%d %d %.17g\n", x, y, a[q]);
      if (r < 0) { ok = false; break; }
    }
    if (ok && std::fputc('\n', f) == EOF) ok = false;
  }
  return std::fclose(f) == 0 && ok;
}
static bool write_profile(const std::string& path, int ny, const double* a) {
  FILE* f = std::fopen(path.c_str(), "w");
  if (!f) return false;
  bool ok = true;
  for (int y = 0; y < ny && ok; y++) ok = std::fprintf(f, "%d %.17g\n", y, a[y]) >= 0;
  return std::fclose(f) == 0 && ok;
}
// "binary VTK 2.0" (L244-246): legacy header, then the values as big-endian doubles (the byte order the legacy format fixes)
static bool write_vtk(const std::string& path, const char* name, int nx, int ny, const double* a, const double* b) {
  FILE* f = std::fopen(path.c_str(), "wb");
  if (!f) return false;
  bool ok = std::fprintf(f, "# vtk DataFile Version 2.0\n%s\nBINARY\nDATASET STRUCTURED_POINTS\nDIMENSIONS %d %d 1\n"
                            "ORIGIN 0 0 0\nSPACING 1 1 1\nPOINT_DATA %lld\n", name, nx, ny, (long long)nx * ny) >= 0;
  if (ok) ok = (b ? std::fprintf(f, "VECTORS %s double\n", name) : std::fprintf(f, "SCALARS %s double 1\nLOOKUP_TABLE default\n", name)) >= 0;
  const size_t n = (size_t)nx * ny, per = b ? 3 : 1;
  std::vector<unsigned char> out;
  try { out.resize(n * per * 8); } catch (...) { std::fclose(f); return false; }
  auto put = [&](size_t slot, double v) {
    uint64_t u;
    std::memcpy(&u, &v, 8);
    for (int k = 0; k < 8; k++) out[slot * 8 + k] = (unsigned char)(u >> (56 - 8 * k));
  };
  for (size_t q = 0; q < n; q++) {
    put(q * per, a[q]);
    if (b) { put(q * per + 1, b[q]); put(q * per + 2, 0.0); }
  }
  if (ok) ok = std::fwrite(out.data(), 1, out.size(), f) == out.size();
  if (ok) ok = std::fputc('\n', f) != EOF;
  return std::fclose(f) == 0 && ok;
}

int tlb_write_fields(tlb_handle* h, const char* dir, int32_t index, int32_t what, int32_t vtk) {
  if (!h || !dir || what < 0 || what > 31) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  const int nx = h->d.nx, ny = h->d.ny;
  const size_t n = (size_t)nx * ny;
  std::vector<double> a, b;
  try { a.resize(2 * n); b.resize((size_t)ny > n ? (size_t)ny : n); } catch (...) { return TLB_EINVAL; }
  const std::string base = std::string(dir) + "/", tag = "." + std::to_string(index);
  auto field = [&](const char* name, const double* p, const double* q) {
    if (!write_dat(base + name + tag + ".dat", nx, ny, p, q)) return false;
    return !vtk || write_vtk(base + name + tag + ".vtk", name, nx, ny, p, q);
  };
  int rc;
  if (what & (TLB_OUT_DENSITY | TLB_OUT_TEMPERATURE | TLB_OUT_VELOCITY)) {
    if (what & TLB_OUT_DENSITY) {
      if ((rc = tlb_fields_host(h, a.data(), b.data(), nullptr, nullptr)) != TLB_OK) return rc;
      if (!field("firstdensity", a.data(), nullptr) || !field("seconddensity", b.data(), nullptr)) return TLB_EIO;
    }
    if (what & TLB_OUT_TEMPERATURE) {
      if ((rc = tlb_fields_host(h, nullptr, nullptr, nullptr, a.data())) != TLB_OK) return rc;
      if (!field("temperature", a.data(), nullptr)) return TLB_EIO;
    }
    if (what & TLB_OUT_VELOCITY) {
      if ((rc = tlb_fields_host(h, nullptr, nullptr, a.data(), nullptr)) != TLB_OK) return rc;
      if (!field("veloconf", a.data(), a.data() + n)) return TLB_EIO;
      if ((rc = tlb_x_average_host(h, b.data())) != TLB_OK) return rc;
      if (!write_profile(base + "u_av" + tag + ".dat", ny, b.data())) return TLB_EIO;
    }
  }
  if (what & TLB_OUT_STRESS) {
    if ((rc = tlb_stress_xy_host(h, a.data())) != TLB_OK) return rc;
    if (!field("Ptot_xy", a.data(), nullptr)) return TLB_EIO;
    if ((rc = tlb_x_average_stress_host(h, b.data())) != TLB_OK) return rc;
    if (!write_profile(base + "Pxy_av" + tag + ".dat", ny, b.data())) return TLB_EIO;
  }
  if (what & TLB_OUT_ENERGY) {  // timeEnergy.dat (L248): one line per call, appended
    double o4[4];
    if ((rc = tlb_observables_host(h, o4)) != TLB_OK) return rc;
    FILE* f = std::fopen((base + "timeEnergy.dat").c_str(), "a");
    if (!f) return TLB_EIO;
    const bool ok = std::fprintf(f, "%d %.17g\n", (int)index, o4[2]) >= 0;
    if (std::fclose(f) != 0 || !ok) return TLB_EIO;
  }
  return TLB_OK;
}

int tlb_step(tlb_handle* h, int64_t n) {
  if (!h || n < 0) return TLB_EINVAL;
  if (h->halo_lo || h->halo_hi) return TLB_EINVAL;  // a slab with halo rows steps through the tlb_slab_step_* calls
  if (!h->has_state) return TLB_ESTATE;
  TLB_ENTER(h);
  // the graphs of both buffer parities are captured on the first call, before anything is enqueued, so that a
  // caller timing a later call never times cudaGraphInstantiate
  if (n > 0 && h->use_graph) { ensure_graph(h, 0); ensure_graph(h, 1); }
  int64_t t = 0;
  // whole blocks of kGraphSteps steps replay a captured graph (one launch instead of 2 * kGraphSteps)
  while (n - t >= kGraphSteps && ensure_graph(h, h->cur)) {
    if (cu(h, cudaGraphLaunch(h->gexec[h->cur], h->st)) != TLB_OK) return TLB_ECUDA;
    h->launches += h->g_launches[h->cur];
    t += kGraphSteps;  // an even number of steps: h->cur is unchanged
  }
  for (; t < n; t++) {
    void* in = h->S[h->cur];
    void* out = h->S[1 - h->cur];
    h->launches += launch_step(h, in, out, h->d.own0, h->d.own1, h->st);
    h->launches += launch_boundary(h->d, out, h->sites, h->n_sites, h->st);
    h->cur = 1 - h->cur;
  }
  return check(h);
}

// ---- y-slab stepping: edges -> (pack, exchange, unpack by the caller) -> interior -> finish ----
static void edge_rows(const tlb_handle* h, int* lo_end, int* hi_beg) {
  const int a = h->d.own0, b = h->d.own1;
  *lo_end = h->halo_lo ? (a + kHalo < b ? a + kHalo : b) : a;
  const int hb = h->halo_hi ? b - kHalo : b;
  *hi_beg = hb > *lo_end ? hb : *lo_end;
}

int tlb_slab_step_edges(tlb_handle* h) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  int lo_end, hi_beg;
  edge_rows(h, &lo_end, &hi_beg);
  h->launches += launch_step(h, h->S[h->cur], h->S[1 - h->cur], h->d.own0, lo_end, h->st);
  h->launches += launch_step(h, h->S[h->cur], h->S[1 - h->cur], hi_beg, h->d.own1, h->st);
  h->step_open = true;
  return check(h);
}

int tlb_slab_step_interior(tlb_handle* h) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || !h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  int lo_end, hi_beg;
  edge_rows(h, &lo_end, &hi_beg);
  h->launches += launch_step(h, h->S[h->cur], h->S[1 - h->cur], lo_end, hi_beg, h->st);
  return check(h);
}

int tlb_slab_step_finish(tlb_handle* h) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || !h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_boundary(h->d, h->S[1 - h->cur], h->sites, h->n_sites, h->st);
  h->cur = 1 - h->cur;
  h->step_open = false;
  return check(h);
}

int tlb_halo_pack(tlb_handle* h, int face, void* buf) {
  if (!h || !buf || face < 0 || face > 1 || !(face ? h->halo_hi : h->halo_lo)) return TLB_EINVAL;
  if (!h->has_state) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_halo_pack(h->d, h->S[h->step_open ? 1 - h->cur : h->cur], face, buf, h->st);
  return check(h);
}

int tlb_halo_unpack(tlb_handle* h, int face, const void* buf) {
  if (!h || !buf || face < 0 || face > 1 || !(face ? h->halo_hi : h->halo_lo)) return TLB_EINVAL;
  if (!h->has_state) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_halo_unpack(h->d, h->S[h->step_open ? 1 - h->cur : h->cur], face, buf, h->st);
  return check(h);
}

int tlb_halo_region(tlb_handle* h, int face, int which, void** ptr, size_t* bytes) {
  if (!h || !ptr || !bytes || face < 0 || face > 1 || which < 0 || which > 1 || !(face ? h->halo_hi : h->halo_lo)) return TLB_EINVAL;
  if (!h->has_state) return TLB_ESTATE;
  const Dev& d = h->d;
  const size_t esz = d.prec == 32 ? sizeof(float) : sizeof(double);
  int y;  // first local row of the block
  if (which == 0) y = face == 0 ? d.own0 : d.own1 - kHalo;
  else y = face == 0 ? d.own0 - kHalo : d.own1;
  char* S = static_cast<char*>(h->S[h->step_open ? 1 - h->cur : h->cur]);
  *ptr = S + (size_t)(y + 1) * (size_t)d.row * esz;  // storage row y + 1; a row holds the 27 plane rows
  *bytes = (size_t)kHalo * (size_t)d.row * esz;
  return TLB_OK;
}

int tlb_profile_step(tlb_handle* h, int64_t n, double* fused_ms, double* boundary_ms) {
  if (!h || n < 1 || n > 4096 || !fused_ms || !boundary_ms) return TLB_EINVAL;
  if (h->halo_lo || h->halo_hi) return TLB_EINVAL;
  if (!h->has_state) return TLB_ESTATE;
  TLB_ENTER(h);
  // Both kernels are idempotent on fixed inputs (the fused kernel reads S[cur] and writes S[1-cur]; the
  // boundary kernel reads fluid nodes and writes solid / ghost nodes), so each is launched n times back
  // to back between two events and the state advances by exactly one step.
  cudaEvent_t ev[3];
  for (auto& e : ev) cu(h, cudaEventCreate(&e));
  void* in = h->S[h->cur];
  void* out = h->S[1 - h->cur];
  cu(h, cudaEventRecord(ev[0], h->st));
  for (int64_t t = 0; t < n; t++) h->launches += launch_step(h, in, out, h->d.own0, h->d.own1, h->st);
  cu(h, cudaEventRecord(ev[1], h->st));
  for (int64_t t = 0; t < n; t++) h->launches += launch_boundary(h->d, out, h->sites, h->n_sites, h->st);
  cu(h, cudaEventRecord(ev[2], h->st));
  h->cur = 1 - h->cur;
  cu(h, cudaStreamSynchronize(h->st));
  float a = 0.f, b = 0.f;
  if (h->err == cudaSuccess) {
    cu(h, cudaEventElapsedTime(&a, ev[0], ev[1]));
    cu(h, cudaEventElapsedTime(&b, ev[1], ev[2]));
  }
  for (auto& e : ev) cudaEventDestroy(e);
  *fused_ms = (double)a / (double)n;
  *boundary_ms = (double)b / (double)n;
  return check(h);
}

// rows the non-stepping modes of the fused kernel sweep: the owned ones
static int fused_mode(tlb_handle* h, int mode, const FusedOut& out) {
  const int seg = default_seg_rows(h->d.nx, h->d.own1 - h->d.own0);
  h->launches += launch_fused(h->d, mode, h->S[h->cur], nullptr, seg, h->d.own0, h->d.own1, out, maps_of(h, h->S[h->cur]), h->st);
  return check(h);
}

static int fields_to_scratch(tlb_handle* h) {
  FusedOut o{};
  o.rhoA = h->fld[0]; o.rhoB = h->fld[1]; o.ux = h->fld[2]; o.uy = h->fld[3]; o.T = h->fld[4];
  return fused_mode(h, 1, o);
}

int tlb_fields(tlb_handle* h, double* rho_A, double* rho_B, double* u, double* T) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  const size_t n = (size_t)h->d.nx * h->d.ny;
  FusedOut o{};
  o.rhoA = rho_A; o.rhoB = rho_B; o.ux = u; o.uy = u ? u + n : nullptr; o.T = T;
  return fused_mode(h, 1, o);
}

int tlb_fields_host(tlb_handle* h, double* rho_A, double* rho_B, double* u, double* T) {
  if (!h) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  const size_t n = (size_t)h->d.nx * h->d.ny, b = n * sizeof(double);
  fields_to_scratch(h);
  if (rho_A) cu(h, cudaMemcpyAsync(rho_A, h->fld[0], b, cudaMemcpyDeviceToHost, h->st));
  if (rho_B) cu(h, cudaMemcpyAsync(rho_B, h->fld[1], b, cudaMemcpyDeviceToHost, h->st));
  if (u) cu(h, cudaMemcpyAsync(u, h->fld[2], 2 * b, cudaMemcpyDeviceToHost, h->st));
  if (T) cu(h, cudaMemcpyAsync(T, h->fld[4], b, cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

// one pass: the fused kernel (MODE 3) reduces inside each CTA, a single small kernel combines the CTAs
static int observable_pass(tlb_handle* h, double* sums6, double* out4) {
  FusedOut o{};
  o.partials = h->partials;
  int rc = fused_mode(h, 3, o);
  if (rc != TLB_OK) return rc;
  h->launches += launch_observables_final(h->d, h->partials, h->obs_ctas, sums6, out4, h->st);
  return check(h);
}

int tlb_observables(tlb_handle* h, double* out4) {
  if (!h || !out4) return TLB_EINVAL;
  if (h->halo_lo || h->halo_hi) return TLB_EINVAL;  // a slab holds part of the sums: tlb_observable_sums
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  return observable_pass(h, nullptr, out4);
}

int tlb_observables_host(tlb_handle* h, double* out4) {
  if (!h || !out4) return TLB_EINVAL;
  int rc = tlb_observables(h, h->out4);
  if (rc != TLB_OK) return rc;
  TLB_ENTER(h);
  cu(h, cudaMemcpyAsync(out4, h->out4, 4 * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

int tlb_observable_sums(tlb_handle* h, double* sums6) {
  if (!h || !sums6) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  return observable_pass(h, sums6, nullptr);
}

int tlb_observables_from_sums(tlb_handle* h, const double* sums6, double* out4) {
  if (!h || !sums6 || !out4) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_observables_from_sums(h->d, sums6, out4, h->st);
  return check(h);
}

int tlb_x_average(tlb_handle* h, double* u_av) {
  if (!h || !u_av) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  fields_to_scratch(h);
  h->launches += launch_x_average(h->d, h->fld[2], u_av, h->st);
  return check(h);
}

int tlb_x_average_host(tlb_handle* h, double* u_av) {
  if (!h || !u_av) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  fields_to_scratch(h);
  // fld[0] (rho_A scratch) is free once the profile has been reduced from fld[2]
  h->launches += launch_x_average(h->d, h->fld[2], h->fld[0], h->st);
  cu(h, cudaMemcpyAsync(u_av, h->fld[0], (size_t)h->d.ny * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

int tlb_stress_xy(tlb_handle* h, double* P_xy) {
  if (!h || !P_xy) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  FusedOut o{};
  o.pxy = P_xy;
  return fused_mode(h, 2, o);
}

int tlb_stress_xy_host(tlb_handle* h, double* P_xy) {
  if (!h || !P_xy) return TLB_EINVAL;
  int rc = tlb_stress_xy(h, h->fld[0]);
  if (rc != TLB_OK) return rc;
  TLB_ENTER(h);
  cu(h, cudaMemcpyAsync(P_xy, h->fld[0], (size_t)h->d.nx * h->d.ny * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

int tlb_x_average_stress(tlb_handle* h, double* Pxy_av) {
  if (!h || !Pxy_av) return TLB_EINVAL;
  int rc = tlb_stress_xy(h, h->fld[0]);
  if (rc != TLB_OK) return rc;
  TLB_ENTER(h);
  h->launches += launch_x_average(h->d, h->fld[0], Pxy_av, h->st);
  return check(h);
}

int tlb_x_average_stress_host(tlb_handle* h, double* Pxy_av) {
  if (!h || !Pxy_av) return TLB_EINVAL;
  int rc = tlb_x_average_stress(h, h->fld[1]);
  if (rc != TLB_OK) return rc;
  TLB_ENTER(h);
  cu(h, cudaMemcpyAsync(Pxy_av, h->fld[1], (size_t)h->d.ny * sizeof(double), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

// Droplet analysis, first stage (section 2.4): scratch planes fld[1..3] hold the labels, the root lists and the sums.
int tlb_droplets(tlb_handle* h, double B_th, int32_t* labels, int32_t max_droplets, int32_t* n_droplets, double* stats) {
  if (!h || !n_droplets || max_droplets < 0 || (max_droplets > 0 && !stats)) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;  // a global analysis: gather the density field of the slabs first
  const size_t n = (size_t)h->d.nx * h->d.ny;
  if ((size_t)max_droplets * 4 > n) return TLB_EINVAL;  // root lists and sums live in scratch planes
  if (!h->has_state) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_rho_a(h->d, h->S[h->cur], h->fld[0], h->st);  // only the first fluid's 9 planes are read
  int* lab = labels ? labels : reinterpret_cast<int*>(h->fld[1]);
  h->launches += launch_label_init(h->d, h->fld[0], B_th, lab, h->st);
  h->launches += launch_label_merge(h->d, lab, h->st);
  h->launches += launch_label_flatten(h->d, lab, h->st);
  int* roots = reinterpret_cast<int*>(h->fld[2]);
  cu(h, cudaMemsetAsync(n_droplets, 0, sizeof(int), h->st));
  if (max_droplets > 0) cu(h, cudaMemsetAsync(h->fld[3], 0, 3 * sizeof(unsigned long long) * (size_t)max_droplets, h->st));
  h->launches += launch_droplet_stats(h->d, lab, roots, roots + max_droplets, reinterpret_cast<unsigned long long*>(h->fld[3]),
                                      max_droplets, n_droplets, stats, h->st);
  return check(h);
}

int tlb_droplets_host(tlb_handle* h, double B_th, int32_t* labels, int32_t max_droplets, int32_t* n_droplets, double* stats) {
  if (!h || !n_droplets || max_droplets < 0 || (max_droplets > 0 && !stats)) return TLB_EINVAL;
  const size_t n = (size_t)h->d.nx * h->d.ny;
  if ((size_t)max_droplets * 4 > n) return TLB_EINVAL;  // device copy of the statistics lives in a scratch plane
  int* lab = reinterpret_cast<int*>(h->fld[1]);
  double* dstats = h->fld[4];
  int rc = tlb_droplets(h, B_th, lab, max_droplets, h->n_drop, dstats);
  if (rc != TLB_OK) return rc;
  TLB_ENTER(h);
  if (labels) cu(h, cudaMemcpyAsync(labels, lab, n * sizeof(int), cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaMemcpyAsync(n_droplets, h->n_drop, sizeof(int), cudaMemcpyDeviceToHost, h->st));
  if (max_droplets > 0) cu(h, cudaMemcpyAsync(stats, dstats, 4 * sizeof(double) * (size_t)max_droplets, cudaMemcpyDeviceToHost, h->st));
  cu(h, cudaStreamSynchronize(h->st));
  return check(h);
}

// ---- droplet analysis, second stage (section 2.4, Eq. (25); readings R23-R26).  Scratch planes fld[2], fld[3]
// hold the cell grid / adjacency tables / events found.
int tlb_voronoi(tlb_handle* h, const double* centres, int32_t n, int32_t* colour) {
  if (!h || !colour || n < 0 || (n > 0 && !centres)) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  const size_t N = (size_t)h->d.nx * h->d.ny;
  if ((size_t)n * 4 > N) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_voronoi(h->d, centres, n, reinterpret_cast<int*>(h->fld[2]), colour, h->st);
  return check(h);
}

int tlb_delaunay(tlb_handle* h, const int32_t* colour, int32_t n, int32_t max_links, int32_t* n_links, int32_t* links) {
  if (!h || !colour || !n_links || n < 0 || max_links < 0 || (max_links > 0 && !links)) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  const size_t N = (size_t)h->d.nx * h->d.ny;
  if ((size_t)n * (kMaxDegree + 1) + 3 > 2 * N) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_delaunay(h->d, colour, n, reinterpret_cast<int*>(h->fld[2]), max_links, n_links, links, h->st);
  return check(h);
}

int tlb_droplet_match(tlb_handle* h, const int32_t* colour_past, const double* centres_now, int32_t n_now, int32_t* map) {
  if (!h || !colour_past || n_now < 0 || (n_now > 0 && (!centres_now || !map))) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_match(h->d, colour_past, centres_now, n_now, map, h->st);
  return check(h);
}

int tlb_droplet_displacements(tlb_handle* h, const double* centres_past, const double* centres_now, const int32_t* map,
                              int32_t n_now, double* disp) {
  if (!h || n_now < 0 || (n_now > 0 && (!centres_past || !centres_now || !map || !disp))) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  TLB_ENTER(h);
  h->launches += launch_displacements(h->d, centres_past, centres_now, map, n_now, disp, h->st);
  return check(h);
}

int tlb_t1_events(tlb_handle* h, const int32_t* links_past, int32_t n_past, const int32_t* links_now, int32_t n_now,
                  const int32_t* map, int32_t n_map, int32_t n_droplets, int32_t max_events, int32_t* n_events,
                  int32_t* events) {
  if (!h || !n_events || n_past < 0 || n_now < 0 || n_droplets < 0 || max_events < 0 || n_map < 0) return TLB_EINVAL;
  if ((n_past > 0 && !links_past) || (n_now > 0 && !links_now) || (max_events > 0 && !events)) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  const size_t N = (size_t)h->d.nx * h->d.ny;
  if (2 * (size_t)n_droplets * kMaxDegree > 2 * N || N < 8) return TLB_EINVAL;
  TLB_ENTER(h);
  // fld[2], fld[3] are adjacent planes: the two tables fill (part of) the first, the events found start at the second
  int* scratch = reinterpret_cast<int*>(h->fld[2]);
  size_t cap = (2 * N - 2) / 4;  // events that fit behind the two counters in fld[3]
  if (cap > (size_t)1 << 20) cap = (size_t)1 << 20;
  // launch_t1 lays the counters and the event list right behind the tables
  h->launches += launch_t1(links_past, n_past, links_now, n_now, map, n_map, n_droplets, scratch, (int)cap, max_events,
                           n_events, events, h->st);
  return check(h);
}

int tlb_droplet_nusselt(tlb_handle* h, const double* centres, int32_t n, double* nu) {
  if (!h || n < 0 || (n > 0 && (!centres || !nu))) return TLB_EINVAL;
  if (h->slab) return TLB_EINVAL;
  if (!h->has_state || h->step_open) return TLB_ESTATE;
  TLB_ENTER(h);
  h->launches += launch_droplet_nusselt(h->d, h->S[h->cur], centres, n, h->p.tau_g, nu, h->st);
  return check(h);
}

int64_t tlb_launch_count(const tlb_handle* h) { return h ? h->launches : 0; }

const char* tlb_error_string(int code) {
  switch (code) {
    case TLB_OK: return "ok";
    case TLB_EINVAL: return "invalid argument (size, parameter, NULL pointer, workspace too small, or a call this kind of handle does not take)";
    case TLB_ESTATE: return "no state (call tlb_init, tlb_set_fields or tlb_set_populations first) or slab step calls out of order";
    case TLB_ECUDA: return "CUDA error (see tlb_last_cuda_error); there is no CPU fallback";
    case TLB_EPLACEMENT: return "tlb_init could not place n_droplets by random sequential addition";
    case TLB_EIO: return "checkpoint file missing, unreadable, unwritable or of another lattice size";
    case TLB_ELIMIT: return "size beyond the fixed capacity of tlb_t1_events_static (TLB_T1_STATIC_MAX_DROPLETS droplets, 64 devices)";
  }
  return "unknown error code";
}

const char* tlb_last_cuda_error(const tlb_handle* h) { return cudaGetErrorString(h ? h->err : cudaSuccess); }

}  // extern "C"
