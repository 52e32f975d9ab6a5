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
// A plane is [ny + 2][px] doubles, x fastest, lattice column x at offset kXL + x within a row; px
// and kXL are multiples of 16 doubles so that x = 0 of every row starts a 128-byte line and the
// strip copies of the fused kernel (cp.async.bulk) are 16-byte aligned.  27 planes per buffer:
// [0, 9) f_A, [9, 18) f_B, [18, 27) g, direction order R1.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tlb.h"

namespace tlb {

// D2Q9 directions in the ABI order (R1).  opp(i) = direction with c = -c_i.
__host__ __device__ constexpr int cx(int i) { return i == 1 || i == 5 || i == 8 ? 1 : (i == 3 || i == 6 || i == 7 ? -1 : 0); }
__host__ __device__ constexpr int cy(int i) { return i == 2 || i == 5 || i == 6 ? 1 : (i == 4 || i == 7 || i == 8 ? -1 : 0); }
__host__ __device__ constexpr int opp(int i) { return i == 0 ? 0 : (i <= 4 ? ((i + 1) % 4) + 1 : ((i - 3) % 4) + 5); }
__host__ __device__ constexpr double wq(int i) { return i == 0 ? 4.0 / 9.0 : (i <= 4 ? 1.0 / 9.0 : 1.0 / 36.0); }

// fused-kernel geometry (see tlb_step.cu)
#ifndef TLB_KW
#define TLB_KW 128
#endif
constexpr int kW = TLB_KW;              // strip width = lattice columns per CTA (two threads per column)
constexpr int kHX = 4;                  // columns fetched beyond the strip on each side (3 needed; 4 keeps 16-byte alignment)
constexpr int kCopyW = kW + 2 * kHX;    // doubles per plane-row copy
constexpr int kSlots = 4;               // rows of the 18 fluid planes resident in shared memory
constexpr int kRingRows = 6;            // rows of rho / psi kept in shared memory
constexpr int kXL = 16;                 // padded-row offset of lattice column 0
constexpr int kGhost = kHX;             // ghost columns kept valid on each side

// Everything a kernel needs, passed by value (lives in the constant bank of the launch).
struct Dev {
  int nx, ny;
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

  // offset of lattice node (x, y) inside a plane; x in [-kXL, px - kXL), y in [-1, ny]
  __host__ __device__ long long at(int x, int y) const { return (long long)(y + 1) * row + kXL + x; }
};

__host__ __device__ inline int padded_pitch(int nx) {
  const int strips = (nx + kW - 1) / kW;
  return kXL + strips * kW + 16;  // multiple of 16; room for the last strip's copy overhang
}

// launchers (each returns the number of kernels it launched)
int launch_step(const Dev& d, const void* Sin, void* Sout, int seg_rows, cudaStream_t st);
int launch_fields(const Dev& d, const void* S, double* rhoA, double* rhoB, double* ux, double* uy, double* T,
                  cudaStream_t st);
int launch_boundary(const Dev& d, void* S, const int* sites, int n_sites, cudaStream_t st);
int launch_build_links(const Dev& d, int* sites, int* count, uint8_t* solidp, cudaStream_t st);
int launch_scatter(const Dev& d, const double* fA, const double* fB, const double* g, void* S, cudaStream_t st);
int launch_gather(const Dev& d, const void* S, double* fA, double* fB, double* g, cudaStream_t st);
int launch_set_fields(const Dev& d, const double* rhoA, const double* rhoB, const double* T, void* S,
                      cudaStream_t st);
int launch_copy_g(const Dev& d, const void* Ssrc, void* Sdst, cudaStream_t st);
int launch_init(const Dev& d, const tlb_params& p, uint64_t seed, const double* centres, int n_centres,
                uint8_t* inside_scratch, uint8_t* solid, double* rhoA, double* rhoB, double* T, cudaStream_t st);
int launch_observables(const Dev& d, const double* rhoA, const double* rhoB, const double* ux, const double* uy,
                       const double* T, double* partials, int n_blocks, double* out4, cudaStream_t st);
int launch_x_average(const Dev& d, const double* ux, double* u_av, cudaStream_t st);
int configure_kernels();  // opt in to the dynamic shared memory the fused kernel needs; 0 on success
int default_seg_rows(int nx, int ny);
constexpr int kObsBlocks = 592; // 4 per SM on 148 SMs

}  // namespace tlb
