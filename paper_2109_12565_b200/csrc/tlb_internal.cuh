// tlb_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
//
// Storage ("pull form"): a population buffer holds S_i(s) = f*_i(s, t-1), the post-collision
// population of the previous step, NOT yet streamed.  The time-t population of PAPER Eq. (1) (L63)
// is then
//     f_i(x, t) = S_i(x - c_i),
// a pure gather.  The lattice is padded so that the gather never needs index arithmetic:
//   * one ghost row below (storage row 0 = lattice row -1) and above (lattice row ny): the boundary
//     kernel stores into every solid / ghost node s the reflected value its fluid neighbour
//     x = s + c_i will pull, S_i(s) = S_opp(i)(x) (half-way bounce-back, L151) and, for g,
//     -S_opp(i)(x) + 2 w_i T_w(s) (R8);
//   * ghost columns x = -kGhost..-1 and nx..nx+kGhost-1 hold the periodic images S(x -+ nx) (the
//     paper's own ghost-node device, footnote 2 L180); every kernel that writes column x also
//     writes its images, so no separate halo-refresh pass exists.
// A buffer is [ny + 2][27][px] doubles: x fastest, then the 27 planes of one row, then the rows ("row-interleaved
// planes"; Dev.plane = px and Dev.row = 27 px are the strides, and nothing but tlb_create fixes them); lattice column
// x sits at offset kXL + x within a plane row; px
// and kXL are multiples of 16 doubles so that x = 0 of every row starts a 128-byte line and the
// strip copies of the fused kernel are 16-byte aligned.  27 planes per buffer: [0, 9) f_A, [9, 18) f_B,
// [18, 27) g; inside a set the planes are ordered by c_y (pslot() below): the three directions with
// c_y = +1, then c_y = 0, then c_y = -1.  A target row r pulls storage row (r + 1) - c_y of plane i, so
// with this order ONE tensor-map copy (cp.async.bulk.tensor, box x * 1 row * 3 planes * 3 groups * 2 species,
// group stride = 3 planes + 1 row) brings the 18 fluid plane rows of a strip, already shifted in y.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <cmath>

#include "../../include/tlb.h"

namespace tlb {

// D2Q9 directions in the ABI order (R1).  opp(i) = direction with c = -c_i.
__host__ __device__ constexpr int cx(int i) { return i == 1 || i == 5 || i == 8 ? 1 : (i == 3 || i == 6 || i == 7 ? -1 : 0); }
__host__ __device__ constexpr int cy(int i) { return i == 2 || i == 5 || i == 6 ? 1 : (i == 4 || i == 7 || i == 8 ? -1 : 0); }
__host__ __device__ constexpr int opp(int i) { return i == 0 ? 0 : (i <= 4 ? ((i + 1) % 4) + 1 : ((i - 3) % 4) + 5); }
// plane of direction i inside its set (internal order, see above); the ABI keeps the order R1
__host__ __device__ constexpr int pslot(int i) {
  return i == 2 ? 0 : i == 5 ? 1 : i == 6 ? 2 : i == 0 ? 3 : i == 1 ? 4 : i == 3 ? 5 : i == 4 ? 6 : i == 7 ? 7 : 8;
}
__host__ __device__ constexpr double wq(int i) { return i == 0 ? 4.0 / 9.0 : (i <= 4 ? 1.0 / 9.0 : 1.0 / 36.0); }

// fused-kernel geometry (see tlb_step.cu)
constexpr int kW = 128;                 // strip width = lattice columns per CTA (two threads per column)
constexpr int kHX = 4;                  // columns fetched beyond the strip on each side (3 needed; 4 keeps 16-byte alignment)
constexpr int kCopyW = kW + 2 * kHX;    // doubles per plane-row copy
constexpr int kSlots = 4;               // rows of the 18 fluid planes resident in shared memory
constexpr int kRingRows = 6;            // rows of rho / psi kept in shared memory
constexpr int kXL = 16;                 // padded-row offset of lattice column 0
constexpr int kGhost = kHX;             // ghost columns kept valid on each side
constexpr int kHalo = 3;                // halo rows per interior face of a y-slab (see tlb.h, "Y-SLABS")

// Everything a kernel needs, passed by value (lives in the constant bank of the launch).
struct Dev {
  int nx, ny;            // local lattice; for a y-slab ny counts the halo rows too
  int y_off, ny_glob;    // y-slab: global row of local row 0 and rows of the whole lattice (else 0, ny)
  int per_glob;          // the whole lattice is periodic in y (a slab of it is not: its faces import halo rows)
  int wall_lo, wall_hi;  // is there a flat wall beyond local row 0 / ny - 1 (else: periodic wrap, or a slab face)
  int own0, own1;        // local rows this handle computes (a slab imports the others from its neighbours)
  int px;                // padded row pitch in doubles (and in bytes of the padded mask)
  int periodic_y, thermal;
  int prec;              // storage precision of the populations: 64 (double) or 32 (float; arithmetic stays fp64)
  long long plane;       // elements between consecutive planes of one node
  long long row;         // elements between consecutive rows of one plane
  double omega, omega_g; // 1/tau, 1/tau_g
  double tau;
  double inv_rho0, rho0;
  double G12, G11a, G11r, G22a, G22r;
  double rho_wall_A, rho_wall_B, pss_wall_A, pss_wall_B; // wall densities and their psi^s (Eq. 12)
  double T_bottom, T_top, T_ref, alpha_g, body_ax;
  double u_wall_bottom, u_wall_top;  // x-velocity of the flat walls (R20)
  const uint8_t* solid;  // [ny][nx]   flag field in the API layout (L286)
  const uint8_t* solidp; // [ny][px]   the same with ghost columns, lattice column x at kXL + x

  // wall temperature carried by a solid node of local row y (R8): lower half of the whole lattice -> T_bottom
  __host__ __device__ int gy(int y) const {  // row of the whole lattice that local row y is
    int g = y + y_off;
    if (per_glob) { g %= ny_glob; if (g < 0) g += ny_glob; }
    return g;
  }
  __host__ __device__ double T_wall(int y) const { return (2 * gy(y) < ny_glob) ? T_bottom : T_top; }
  // offset of lattice node (x, y) inside a plane; x in [-kXL, px - kXL), y in [-1, ny]
  __host__ __device__ long long at(int x, int y) const { return (long long)(y + 1) * row + kXL + x; }
};

__host__ __device__ inline int padded_pitch(int nx) {
  const int strips = (nx + kW - 1) / kW;
  return kXL + strips * kW + 16;  // multiple of 16; room for the last strip's copy overhang
}

// outputs of the fused kernel's non-stepping modes (any pointer may be null)
struct FusedOut {
  double *rhoA, *rhoB, *ux, *uy, *T;  // MODE 1: [ny][nx] planes
  double* pxy;                        // MODE 2
  double* partials;                   // MODE 3: [CTAs][6] {mass_A, mass_B, sum |u|^2, sum u_y T, sum d_y T, fluid sites}
};

// Tensor maps of one population buffer (built by tlb_create with cuTensorMapEncodeTiled; box width = the slot row pitch:
// kCopyW doubles, or kCopyW + 8 floats):
//   f: 5-D (x, row, plane-in-group 3, c_y group 3, species 2), strides (1, row, plane, 3 plane + row, 9 plane);
//   g: 4-D, the same without the species dimension, based at plane 18.
// Row coordinate r addresses, in group k (c_y = 1 - k), storage row r + k = (r + 1) - c_y.
struct TMaps {
  CUtensorMap f, g;
};

// launchers (each returns the number of kernels it launched)
// maps: the tensor maps of the buffer Sin
int launch_fused(const Dev& d, int mode, const void* Sin, void* Sout, int seg_rows, int ya, int yb, const FusedOut& out,
                 const TMaps* maps, cudaStream_t st);
int fused_grid_ctas(const Dev& d, int seg_rows, int rows);  // CTAs launch_fused uses for `rows` rows
int launch_boundary(const Dev& d, void* S, const int* sites, int n_sites, cudaStream_t st);
int launch_build_links(const Dev& d, int* sites, int* count, uint8_t* solidp, cudaStream_t st);
int launch_scatter(const Dev& d, const double* fA, const double* fB, const double* g, void* S, cudaStream_t st);
int launch_gather(const Dev& d, const void* S, double* fA, double* fB, double* g, cudaStream_t st);
int launch_set_fields(const Dev& d, const double* rhoA, const double* rhoB, const double* T, void* S,
                      cudaStream_t st);
int launch_copy_g(const Dev& d, const void* Ssrc, void* Sdst, cudaStream_t st);
int launch_init(const Dev& d, const tlb_params& p, uint64_t seed, const double* centres, int n_centres,
                uint8_t* inside_scratch, uint8_t* solid, double* rhoA, double* rhoB, double* T, cudaStream_t st);
int launch_observables_final(const Dev& d, const double* partials, int n_blocks, double* sums6, double* out4, cudaStream_t st);
int launch_observables_from_sums(const Dev& d, const double* sums6, double* out4, cudaStream_t st);
int launch_x_average(const Dev& d, const double* plane, double* av, cudaStream_t st);
int launch_halo_pack(const Dev& d, const void* S, int face, void* buf, cudaStream_t st);
int launch_halo_unpack(const Dev& d, void* S, int face, const void* buf, cudaStream_t st);
int launch_rho_a(const Dev& d, const void* S, double* rhoA, cudaStream_t st);
int launch_label_init(const Dev& d, const double* rhoA, double threshold, int* labels, cudaStream_t st);
int launch_label_merge(const Dev& d, int* labels, cudaStream_t st);
int launch_label_flatten(const Dev& d, int* labels, cudaStream_t st);
int launch_droplet_stats(const Dev& d, const int* labels, int* roots, int* sorted, unsigned long long* sums,
                         int max_droplets, int* n_out, double* stats, cudaStream_t st);
// droplet analysis, second stage (tlb_analysis.cu)
constexpr int kMaxDegree = 32;  // slots per droplet in the adjacency tables (a Delaunay vertex has 6 links on average)
struct VorGrid {                // uniform grid of cells the centres are binned into
  int gx, gy;
  double inv_wx, inv_wy, wmin;  // 1 / cell width in x and y, the smaller width
};
VorGrid make_vor_grid(int nx, int ny, int n);
int launch_voronoi(const Dev& d, const double* centres, int n, int* scratch, int* colour, cudaStream_t st);
int launch_delaunay(const Dev& d, const int* colour, int n, int* scratch, int max_links, int* n_links, int* links,
                    cudaStream_t st);
int launch_match(const Dev& d, const int* colour_past, const double* centres_now, int n_now, int* map, cudaStream_t st);
int launch_displacements(const Dev& d, const double* past, const double* now, const int* map, int n, double* disp, cudaStream_t st);
int launch_t1(const int* past, int n_past, const int* now, int n_now, const int* map, int n_map, int n, int* scratch, int cap,
              int max_events, int* n_events, int* events, cudaStream_t st);
int launch_droplet_nusselt(const Dev& d, const void* S, const double* centres, int n, double tau_g, double* nu, cudaStream_t st);
int launch_rough_walls(const Dev& d, const int* cut, int height, int up, int down, int width, int lambda, int asymmetric,
                       uint8_t* solid, cudaStream_t st);
int launch_perturb(const Dev& d, double amplitude, double* fA, double* fB, cudaStream_t st);
int configure_kernels();  // opt in to the dynamic shared memory the fused kernel needs; 0 on success
int default_seg_rows(int nx, int ny);

}  // namespace tlb
