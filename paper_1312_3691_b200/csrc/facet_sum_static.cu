// facet_sum_static.cu -- tpmc_facet_sum_static: the a7 reduction F = sum_f P_f for callers that cannot
// allocate device memory.
//
// Who that is: a host program that has handed the whole of the GPU's memory to its own pool, so that a cudaMalloc made
// behind its back fails or eats into what it budgeted; a control loop with a deadline, for which cudaMalloc/cudaFree are
// off limits because they take driver locks and may wait for the whole device to go idle; and code that runs while
// another thread has a stream capture open in the global capture mode, during which the runtime refuses cudaMalloc.
// tpmc_run keeps the partial sums of this reduction in memory that belongs to the mesh handle (cudaMalloc in
// ensure_scratch); the variant below keeps them in an array that is part of the library image instead, so the call itself
// allocates nothing -- no cudaMalloc, no cudaFree, no library routine that allocates.
//
// The price, stated once: every GPU that loads libtpmc.so holds the kScratchBytes (49 408) bytes of the array until the
// process exits, there is ONE array per GPU shared by every call, and inputs larger than TPMC_STATIC_MAX_FACETS are
// refused (TPMC_ECAPACITY), not split.
#include <mutex>

#include "common.cuh"

namespace {

constexpr int kBlock = 256;                       // threads per block
constexpr long long kFacetsPerPart = 4096;        // facets reduced by one block (fixed: the sum's shape depends on nt only)
constexpr int kMaxParts = 2048;                   // capacity of the scratch: partial sums
constexpr int kTicketWords = 32;                  // 256 bytes behind the partial sums, word 0 = the arrival counter
constexpr size_t kScratchDoubles = 3 * (size_t)kMaxParts + kTicketWords;
constexpr size_t kScratchBytes = kScratchDoubles * sizeof(double);
static_assert((long long)kMaxParts * kFacetsPerPart == TPMC_STATIC_MAX_FACETS, "header and scratch capacity disagree");
constexpr int kMaxDevices = 64;

// The scratch: [3 * kMaxParts] partial sums (x, y, z of part p at 3p..3p+2), then the arrival counter.
// In HOST code `g_scratch` is only a handle for the runtime's symbol calls, not a device address: it must never be handed
// to a kernel as a pointer.  Host code gets the address from cudaGetSymbolAddress (scratch_of below).
static __device__ __align__(256) double g_scratch[kScratchDoubles];

// One block sums kFacetsPerPart facets by a fixed tree and stores its partial sum; the block that arrives last adds the
// partial sums by a second fixed tree, writes the force and leaves the counter at zero.  Deterministic for given P, nt.
__global__ void __launch_bounds__(kBlock) k_facet_sum_static(const double* __restrict__ P, long long nt,
                                                             double* scratch, double* __restrict__ force) {
  __shared__ double s[3][kBlock];
  __shared__ bool last;
  double* parts = scratch;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + 3 * (size_t)kMaxParts);
  const long long b = (long long)blockIdx.x * kFacetsPerPart, e = min(nt, b + kFacetsPerPart);
  double acc[3] = {0.0, 0.0, 0.0};
  for (long long f = b + threadIdx.x; f < e; f += kBlock)
    for (int a = 0; a < 3; ++a) acc[a] += P[3 * f + a];
  for (int a = 0; a < 3; ++a) s[a][threadIdx.x] = acc[a];
  __syncthreads();
  for (int st = kBlock / 2; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st)
      for (int a = 0; a < 3; ++a) s[a][threadIdx.x] += s[a][threadIdx.x + st];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    for (int a = 0; a < 3; ++a) __stcg(&parts[3 * blockIdx.x + a], s[a][0]);
    __threadfence();   // the partial sum is visible before the arrival is
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();     // every other block's partial sum is visible from here on
  for (int a = 0; a < 3; ++a) acc[a] = 0.0;
  for (int p = threadIdx.x; p < (int)gridDim.x; p += kBlock)
    for (int a = 0; a < 3; ++a) acc[a] += __ldcg(&parts[3 * p + a]);
  for (int a = 0; a < 3; ++a) s[a][threadIdx.x] = acc[a];
  __syncthreads();
  for (int st = kBlock / 2; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st)
      for (int a = 0; a < 3; ++a) s[a][threadIdx.x] += s[a][threadIdx.x + st];
    __syncthreads();
  }
  if (threadIdx.x < 3) force[threadIdx.x] = s[threadIdx.x][0];
  if (threadIdx.x == 0) *ticket = 0u;
}

// Set-up, once per device, with that device current: ask the runtime where this device's copy of g_scratch lives.
std::mutex g_setup_lock;
double* g_scratch_addr[kMaxDevices] = {};

int scratch_of(int device, double** out) {
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_scratch_addr[device]) {
    double* p = nullptr;
    TPMC_CUDA_TRY(cudaGetSymbolAddress((void**)&p, g_scratch));
    if (!p) {
      snprintf(g_tpmc_cuda_error, sizeof(g_tpmc_cuda_error), "cudaGetSymbolAddress(g_scratch) gave no address on device %d", device);
      return TPMC_ECUDA;
    }
    g_scratch_addr[device] = p;
  }
  *out = g_scratch_addr[device];
  return TPMC_OK;
}

}  // namespace

extern "C" int tpmc_facet_sum_static(const double* d_facet_momentum, int64_t nt, void* cuda_stream, double* d_force) {
  if (!d_force || nt < 0 || (nt > 0 && !d_facet_momentum)) return TPMC_EINVAL;
  if (nt > TPMC_STATIC_MAX_FACETS) {
    snprintf(g_tpmc_cuda_error, sizeof(g_tpmc_cuda_error),
             "tpmc_facet_sum_static: nt = %lld exceeds TPMC_STATIC_MAX_FACETS = %lld (fixed scratch of %zu bytes)",
             (long long)nt, (long long)TPMC_STATIC_MAX_FACETS, kScratchBytes);
    return TPMC_ECAPACITY;
  }
  int device = -1;
  TPMC_CUDA_TRY(cudaGetDevice(&device));
  if (device < 0 || device >= kMaxDevices) return TPMC_EINVAL;
  double* scratch = nullptr;
  const int rc = scratch_of(device, &scratch);
  if (rc != TPMC_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // The array keeps what the last call left in it.  The partial sums are all rewritten before they are read; the arrival
  // counter must start at zero, and a call that was cut short could have left it elsewhere: clear it every time.
  TPMC_CUDA_TRY(cudaMemsetAsync(scratch + 3 * (size_t)kMaxParts, 0, sizeof(unsigned int), st));
  const unsigned int parts = nt == 0 ? 1u : (unsigned int)((nt + kFacetsPerPart - 1) / kFacetsPerPart);
  k_facet_sum_static<<<parts, kBlock, 0, st>>>(d_facet_momentum, (long long)nt, scratch, d_force);
  TPMC_CUDA_TRY(cudaGetLastError());
  return TPMC_OK;
}
