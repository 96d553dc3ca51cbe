// peaks.cu -- tpmc_measure_peaks: micro-benchmarks of the units that bound the kernels of the path, measured on the
// device the library runs on ("FP32 = SMs x 128 lanes x clock measured under this load; L2
// and fp64 from micro-benchmarks").  bench.py reports roofline fractions against these numbers, not against products
// of nominal figures.  Each kernel is launched once to warm up and timed once with CUDA events on the caller's stream.
#include "common.cuh"

namespace {

// fp32 lane-instruction issue rate: 8 independent FFMA chains per thread, full occupancy
__global__ void __launch_bounds__(256) k_peak_ffma(float* __restrict__ out, int iters, float a, float b) {
  float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
      x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void __launch_bounds__(256) k_peak_dfma(double* __restrict__ out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1., x2 = x0 + 2., x3 = x0 + 3.;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) { x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b); }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = (x0 + x1) + (x2 + x3);
}

__device__ __forceinline__ unsigned int mix32(unsigned int x) {
  x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
  return x;
}

__global__ void k_peak_fill(uint4* __restrict__ buf, unsigned int n_rec) {
  const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_rec) return;
  // the record a dependent walk visits next: a permutation of the records (multiplier coprime to n_rec), so that
  // walks never merge onto common records
  const unsigned int nx = (unsigned int)(((unsigned long long)i * 1000003ull + 7919ull) % n_rec);
  buf[2 * (size_t)i] = make_uint4(nx, i, 0u, 0u);
  buf[2 * (size_t)i + 1] = make_uint4(0u, 0u, 0u, 0u);
}

// 32-byte read-only gathers (one 256-bit load per lane, every lane its own record) over an array the size of the
// hierarchy, with the traversal kernel's residency (128 threads per block, launch bounds for 8 blocks per SM).
// dependent = 0: the address of load k does not depend on load k-1 (throughput of the L1TEX / L2 gather path);
// dependent = 1: it is read from the record just loaded (the pointer chase of a tree walk: latency x resident warps).
__global__ void __launch_bounds__(128, 8) k_peak_gather(const uint4* __restrict__ buf, unsigned int n_rec, int iters,
                                                        int dependent, unsigned int* __restrict__ out) {
  const unsigned int tid = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int idx = mix32(tid) % n_rec, acc = 0u;
  for (int k = 0; k < iters; ++k) {
    uint4 a, b;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w)
                 : "l"(buf + 2 * (size_t)idx));
    acc ^= a.y ^ b.w;
    idx = dependent ? a.x : mix32(tid + 0x9E3779B9u * (unsigned int)(k + 1)) % n_rec;
  }
  out[tid] = acc;
}

// The traversal kernel's own access shape: a 64-byte record (one wide node) fetched as the two 32-byte halves of one
// line, every lane its own record, at that kernel's residency (128 threads per block, 7 blocks per SM) -- and with two
// records (four loads) in flight per lane before the first result is used, so that the figure is the throughput of the
// L1TEX / L2 gather path and not resident lanes x 32 B / latency, which is what one load in flight per lane measures
// (k_peak_gather above: its independent and dependent variants come out equal for that reason).
__global__ void __launch_bounds__(128, 7) k_peak_gather64(const uint4* __restrict__ buf, unsigned int n_rec64, int iters,
                                                          unsigned int* __restrict__ out) {
  const unsigned int tid = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int acc = 0u;
  for (int k = 0; k < iters; ++k) {
    const unsigned int i0 = mix32(tid + 0x9E3779B9u * (unsigned int)(2 * k + 1)) % n_rec64;
    const unsigned int i1 = mix32(tid + 0x9E3779B9u * (unsigned int)(2 * k + 2)) % n_rec64;
    uint4 a[4], b[4];
    const uint4* p0 = buf + 4 * (size_t)i0;
    const uint4* p1 = buf + 4 * (size_t)i1;
#define TPMC_LD256(A, B, P)                                                                                          \
  asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"                                                \
               : "=r"(A.x), "=r"(A.y), "=r"(A.z), "=r"(A.w), "=r"(B.x), "=r"(B.y), "=r"(B.z), "=r"(B.w)              \
               : "l"(P))
    TPMC_LD256(a[0], b[0], p0);
    TPMC_LD256(a[1], b[1], p0 + 2);
    TPMC_LD256(a[2], b[2], p1);
    TPMC_LD256(a[3], b[3], p1 + 2);
#undef TPMC_LD256
    acc ^= (a[0].y ^ b[0].w) ^ (a[1].y ^ b[1].w) ^ (a[2].y ^ b[2].w) ^ (a[3].y ^ b[3].w);
  }
  out[tid] = acc;
}

// fp64 atomic adds without return value (red.global.add.f64), spread over n_addr accumulators 24 bytes apart
__global__ void __launch_bounds__(256) k_peak_red(double* __restrict__ acc, unsigned int n_addr, int iters) {
  const unsigned int tid = blockIdx.x * blockDim.x + threadIdx.x;
  for (int k = 0; k < iters; ++k) {
    const unsigned int a = mix32(tid * 31u + (unsigned int)k) % n_addr;
    atomicAdd(acc + 3 * (size_t)a, 1.0);
  }
}

struct Timer {
  cudaEvent_t e0, e1;
  cudaStream_t st;
  int init(cudaStream_t s) {
    st = s;
    TPMC_CUDA_TRY(cudaEventCreate(&e0));
    TPMC_CUDA_TRY(cudaEventCreate(&e1));
    return TPMC_OK;
  }
  ~Timer() { cudaEventDestroy(e0); cudaEventDestroy(e1); }
};

}  // namespace

#define PEAK_TIMED(ms_out, launch)                          \
  do {                                                      \
    launch;                                                 \
    TPMC_CUDA_TRY(cudaEventRecord(tm.e0, st));              \
    launch;                                                 \
    TPMC_CUDA_TRY(cudaEventRecord(tm.e1, st));              \
    TPMC_CUDA_TRY(cudaStreamSynchronize(st));               \
    float _ms = 0.f;                                        \
    TPMC_CUDA_TRY(cudaEventElapsedTime(&_ms, tm.e0, tm.e1)); \
    ms_out = _ms;                                           \
  } while (0)

extern "C" int tpmc_measure_peaks(tpmc_peaks* out, void* cuda_stream) {
  if (!out) return TPMC_EINVAL;
  memset(out, 0, sizeof(*out));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0, khz = 0;
  TPMC_CUDA_TRY(cudaGetDevice(&dev));
  TPMC_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  TPMC_CUDA_TRY(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  out->sms = sms;
  out->sm_clock_mhz_nominal = khz * 1e-3;
  Timer tm;
  int rc = tm.init(st);
  if (rc != TPMC_OK) return rc;
  const size_t gather_bytes = (size_t)83 << 20;                 // the size of the C5 hierarchy + facets
  const unsigned int n_rec = (unsigned int)(gather_bytes / 32);
  const unsigned int red_max = 1000000u;
  void *d_out = nullptr, *d_buf = nullptr, *d_acc = nullptr;
  const int nthreads = sms * 16 * 256;
  TPMC_CUDA_TRY(cudaMalloc(&d_out, sizeof(double) * nthreads));
  cudaError_t e = cudaMalloc(&d_buf, gather_bytes);
  if (e == cudaSuccess) e = cudaMalloc(&d_acc, sizeof(double) * 3 * red_max);
  if (e != cudaSuccess) { cudaFree(d_out); cudaFree(d_buf); cudaGetLastError(); return TPMC_ENOMEM; }
  int ret = [&]() -> int {
    float ms;
    {   // fp32: 64 FFMA per loop iteration and thread
      const int iters = 4096;
      PEAK_TIMED(ms, (k_peak_ffma<<<sms * 16, 256, 0, st>>>((float*)d_out, iters, 1.0000001f, 1e-9f)));
      out->fp32_lane_ops_per_s = (double)nthreads * iters * 64.0 / (ms * 1e-3);
      out->sm_clock_mhz_fp32 = out->fp32_lane_ops_per_s / ((double)sms * 128.0) * 1e-6;   // if all 128 lanes issue every cycle
    }
    {   // fp64: 32 DFMA per iteration and thread
      const int iters = 512;
      PEAK_TIMED(ms, (k_peak_dfma<<<sms * 16, 256, 0, st>>>((double*)d_out, iters, 1.0000001, 1e-9)));
      out->fp64_fma_per_s = (double)nthreads * iters * 32.0 / (ms * 1e-3);
    }
    k_peak_fill<<<(n_rec + 255) / 256, 256, 0, st>>>((uint4*)d_buf, n_rec);
    for (int dep = 0; dep < 2; ++dep) {
      const int iters = dep ? 256 : 1024, blocks = sms * 8;
      PEAK_TIMED(ms, (k_peak_gather<<<blocks, 128, 0, st>>>((const uint4*)d_buf, n_rec, iters, dep, (unsigned int*)d_out)));
      const double loads = (double)blocks * 128.0 * iters;
      (dep ? out->gather32_dependent_bytes_per_s : out->gather32_bytes_per_s) = loads * 32.0 / (ms * 1e-3);
    }
    {   // 64-byte records, the traversal kernel's shape and residency
      const int iters = 512, blocks = sms * 7;
      PEAK_TIMED(ms, (k_peak_gather64<<<blocks, 128, 0, st>>>((const uint4*)d_buf, n_rec / 2, iters, (unsigned int*)d_out)));
      out->gather64_bytes_per_s = (double)blocks * 128.0 * iters * 128.0 / (ms * 1e-3);   // 2 records x 64 B per iteration
    }
    out->gather_array_bytes = (double)gather_bytes;
    const unsigned int n_addr[3] = {1u, 2048u, red_max};
    for (int k = 0; k < 3; ++k) {
      const int iters = k == 0 ? 16 : 128, blocks = sms * 8;
      TPMC_CUDA_TRY(cudaMemsetAsync(d_acc, 0, sizeof(double) * 3 * red_max, st));
      PEAK_TIMED(ms, (k_peak_red<<<blocks, 256, 0, st>>>((double*)d_acc, n_addr[k], iters)));
      out->red_f64_per_s[k] = (double)blocks * 256.0 * iters / (ms * 1e-3);
      out->red_f64_addresses[k] = n_addr[k];
    }
    TPMC_CUDA_TRY(cudaGetLastError());
    return TPMC_OK;
  }();
  cudaFree(d_out); cudaFree(d_buf); cudaFree(d_acc);
  return ret;
}
