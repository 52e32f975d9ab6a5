// tlb_noalloc.cu -- tlb_t1_events_static: the T1 search of PAPER section 2.4 (L198-200, reading R25) for callers that
// have no device memory to lend and may not ask CUDA for any.
//
// Everything else in this library works inside the workspace the caller hands to tlb_create; tlb_t1_events keeps its two
// adjacency tables and its list of candidate events in the spare planes of that workspace.  That leaves out whoever
// wants the T1 events of two link lists and has neither a handle nor the right to allocate: a post-processing tool
// in the manner of the paper's deltaAnalysis (L338-341) that only ever reads Delaunay files; a monitor hook that runs
// while the time loop of a lattice sized to fill the GPU is in flight, where cudaMalloc may simply fail and, when it
// succeeds, stalls every stream of the device while it runs; a plug-in living in a host application that hands out
// device memory from its own pool and forbids going around it.  For them the tables live in the array below, which is
// part of the library image: every GPU that loads libtlb.so carries its kTotalInts * 4 bytes (about 4.3 MB) from the
// first CUDA call of the process to its exit, whether or not this entry point is ever called.
//
// The kernels are the ones tlb_t1_events launches (tlb::launch_t1, tlb_analysis.cu); only the scratch differs, so the
// two paths return the same events bit for bit.
#include <mutex>

#include "tlb_internal.cuh"

// adjacency table of the past frame | of the present frame | overflow flag, event counter | candidate events (a, b, c, d)
static constexpr size_t kTableInts = (size_t)TLB_T1_STATIC_MAX_DROPLETS * tlb::kMaxDegree;
static constexpr size_t kTotalInts = 2 * kTableInts + 2 + 4 * (size_t)TLB_T1_STATIC_MAX_EVENTS;

// In host code this name is only a handle for the runtime's symbol calls; it is NOT the device address (a kernel given
// `tlb_t1_static_scratch` from the host side would read host memory or fault).  scratch_of() below asks the runtime for
// the address the array has on the current device.
static __device__ __align__(256) int tlb_t1_static_scratch[kTotalInts];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_lock;
int* g_scratch[kMaxDevices] = {};  // device address of the array, per device ordinal; filled on first use

// Address of the array on the calling thread's current device.  The first call on a device loads the library's
// device code there and looks the symbol up (once; later calls only read the table).
cudaError_t scratch_of(int device, int** out) {
  std::lock_guard<std::mutex> guard(g_lock);
  if (!g_scratch[device]) {
    int* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), tlb_t1_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch[device] = p;
  }
  *out = g_scratch[device];
  return cudaSuccess;
}

}  // namespace

extern "C" int tlb_t1_events_static(const int32_t* links_past, int32_t n_past, const int32_t* links_now, int32_t n_now,
                                    const int32_t* map, int32_t n_map, int32_t n_droplets, int32_t max_events,
                                    int32_t* n_events, int32_t* events, void* stream) {
  if (!n_events || n_past < 0 || n_now < 0 || n_droplets < 0 || max_events < 0 || n_map < 0) return TLB_EINVAL;
  if ((n_past > 0 && !links_past) || (n_now > 0 && !links_now) || (max_events > 0 && !events)) return TLB_EINVAL;
  if (n_droplets > TLB_T1_STATIC_MAX_DROPLETS) return TLB_ELIMIT;  // the tables would not fit the array
  int device = -1;
  if (cudaGetDevice(&device) != cudaSuccess) return TLB_ECUDA;
  if (device < 0 || device >= kMaxDevices) return TLB_ELIMIT;
  if (cudaPeekAtLastError() != cudaSuccess) return TLB_ECUDA;  // somebody else's pending error: not ours to consume
  int* scratch = nullptr;
  if (scratch_of(device, &scratch) != cudaSuccess) { (void)cudaGetLastError(); return TLB_ECUDA; }
  // launch_t1 lays out [n][kMaxDegree] x 2 | overflow, count | [cap][4] from `scratch` on and clears, on the stream, the
  // tables and the two counters before it uses them; the candidate list needs no clearing (only its first `count`
  // entries are read).  Whatever an earlier call left in the array is therefore never seen.
  tlb::launch_t1(links_past, n_past, links_now, n_now, map, n_map, n_droplets, scratch, TLB_T1_STATIC_MAX_EVENTS, max_events,
                 n_events, events, static_cast<cudaStream_t>(stream));
  return cudaGetLastError() == cudaSuccess ? TLB_OK : TLB_ECUDA;
}
