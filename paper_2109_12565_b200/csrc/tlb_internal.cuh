// tlb_internal.cuh -- shared declarations of the CUDA path (never included by oracle/).
//
// Storage ("pull form"): a population buffer holds S_i(s) = f*_i(s, t-1), the post-collision
// population of the previous step, NOT yet streamed, on a lattice padded by one ghost row below
// (row 0) and above (row ny+1).  The time-t population of PAPER Eq. (1) (L63) is then
//     f_i(x, t) = S_i(x - c_i),
// a pure gather.  The boundary kernel makes that gather valid across walls and obstacles by
// storing into every solid / ghost node s the reflected value its fluid neighbour x = s + c_i will
// pull: S_i(s) = S_opp(i)(x) (half-way bounce-back, L151) and, for g, -S_opp(i)(x) + 2 w_i T_w(s)
// (R8).  Planes are [set][i][row][x], x fastest, plane stride (ny+2)*nx doubles.
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

// Everything a kernel needs, passed by value (lives in the constant bank of the launch).
struct Dev {
  int nx, ny;
  int periodic_y, thermal;
  long long plane;       // (ny + 2) * nx, doubles per population plane
  double omega, omega_g; // 1/tau, 1/tau_g
  double tau;
  double inv_rho0, rho0;
  double G12, G11a, G11r, G22a, G22r;
  double rho_wall_A, rho_wall_B, pss_wall_A, pss_wall_B; // wall densities and their psi^s (Eq. 12)
  double T_bottom, T_top, T_ref, alpha_g, body_ax;
  const uint8_t* solid;  // [ny][nx]
};

// strip-marching fused kernel geometry (see tlb_step.cu)
constexpr int kStripThreads = 128;              // threads per CTA = columns incl. halo
constexpr int kHalo = 4;                        // halo columns per side (2 needed; 4 keeps sectors aligned)
constexpr int kStripW = kStripThreads - 2 * kHalo; // interior columns per strip
constexpr int kRing = 6;                        // rows of rho / psi kept in shared memory

struct Links {           // boundary-link work list built by tlb_set_solid
  const int* sites;      // solid in-domain sites that touch fluid, as y * nx + x
  const int* count;      // device counter
};

// launchers (each returns the number of kernels it launched, or sets *err)
int launch_step(const Dev& d, const double* Sin, double* Sout, int seg_rows, cudaStream_t st);
int launch_fields(const Dev& d, const double* S, double* rhoA, double* rhoB, double* ux, double* uy, double* T,
                  cudaStream_t st);
int launch_boundary(const Dev& d, double* S, const int* sites, int n_sites, cudaStream_t st);
int launch_build_links(const Dev& d, int* sites, int* count, cudaStream_t st);
int launch_scatter(const Dev& d, const double* fA, const double* fB, const double* g, double* S, cudaStream_t st);
int launch_gather(const Dev& d, const double* S, double* fA, double* fB, double* g, cudaStream_t st);
int launch_set_fields(const Dev& d, const double* rhoA, const double* rhoB, const double* T, double* S,
                      cudaStream_t st);
int launch_copy_g(const Dev& d, const double* Ssrc, double* Sdst, cudaStream_t st);
int launch_init(const Dev& d, const tlb_params& p, uint64_t seed, const double* centres, int n_centres,
                uint8_t* inside_scratch, uint8_t* solid, double* rhoA, double* rhoB, double* T, cudaStream_t st);
int launch_observables(const Dev& d, const double* rhoA, const double* rhoB, const double* ux, const double* uy,
                       const double* T, double* partials, int n_blocks, double* out4, cudaStream_t st);
constexpr int kObsBlocks = 592; // 4 per SM on 148 SMs

}  // namespace tlb
