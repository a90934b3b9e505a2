// gsr_norm2_static: the two-stage norm of an LSQR vector (row a4: "beta two-stage deterministic
// reduce"; the norms of Algorithm 3) for callers that must not allocate.
//
// Every other entry point of this library takes its scratch memory from a handle, and the handle
// takes it from cudaMalloc.  Some callers cannot do that:
//   - a monitor that checks ||r|| or ||x|| while a config-3-sized solve is resident has almost no
//     free HBM to ask for (the handle holds ~64 GB of tiles plus the work vectors, and a framework
//     around it, e.g. PyTorch's caching allocator, may own whatever is left), so cudaMalloc can
//     fail, or succeed only after the framework has been forced to give its cache back;
//   - cudaMalloc and cudaFree synchronise the whole device, so a call made from a second thread or
//     stream would stall the iteration that is in flight.
// For them this file keeps the scratch of the reduction in a fixed array that is part of the
// loaded library image: STATIC_BYTES (~33 KB) of device memory on every GPU that loads
// libgsr_b200.so, held until the process exits, never allocated or freed by a call.
//
// The array is shared by all calls on a device.  Two calls that may overlap on the GPU (different
// streams without an event between them, or two host threads) race on it and return garbage;
// calls on one stream are safe.  Nothing in it needs to survive from call to call: the ticket
// word is cleared at the start of every call, and the partial sums a call reads are the ones it
// wrote itself (stale ones from a longer, earlier vector lie beyond what it reads).
#include <mutex>

#include "gsr_internal.h"

namespace gsr {

constexpr int SN_TB = 256;                       // threads per CTA
constexpr int SN_PER_THREAD = 512;               // elements per thread
constexpr int64_t SN_CHUNK = (int64_t)SN_TB * SN_PER_THREAD;   // 2^17 elements per CTA
constexpr int SN_MAX_PARTS = 4096;               // partial sums the array can hold
constexpr int SN_HEAD = 32;                      // doubles before the partials: word 0 = ticket
static_assert(SN_CHUNK * SN_MAX_PARTS == GSR_NORM2_STATIC_MAX_LEN, "gsr.h states the limit");
constexpr size_t STATIC_BYTES = (size_t)(SN_HEAD + SN_MAX_PARTS) * 8;
static_assert(STATIC_BYTES == 33024, "gsr.h and README.md state the size of the array");

// The scratch itself.  In DEVICE code this name is the array.  In HOST code it is only a stand-in
// symbol: its host address is not a device address and must never be handed to a kernel (the kernel
// would fault, or on a system where the GPU can reach host memory quietly use the wrong bytes).
// static_scratch_ptr() below turns it into the real address, once per device.
static __device__ __align__(256) double g_static_scratch[SN_HEAD + SN_MAX_PARTS];

// One launch.  CTA c sums the squares of elements [c*SN_CHUNK, (c+1)*SN_CHUNK) in a fixed order
// and stores the partial sum; the CTA that draws the last ticket adds the partials in index
// order and writes sqrt.  The result does not depend on the number of SMs or on which CTA
// finishes last, so equal input gives bit-equal output.
__global__ void __launch_bounds__(SN_TB) k_norm2_static(const double* __restrict__ v, int64_t len,
                                                        double* __restrict__ scratch,
                                                        double* __restrict__ out) {
    __shared__ double red[SN_TB / 32];
    __shared__ int last;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* parts = scratch + SN_HEAD;
    const int64_t i0 = (int64_t)blockIdx.x * SN_CHUNK + threadIdx.x;
    const int64_t i1 = min(len, ((int64_t)blockIdx.x + 1) * SN_CHUNK);
    double q0 = 0.0, q1 = 0.0, q2 = 0.0, q3 = 0.0;
    int64_t i = i0;
    for (; i + 3 * SN_TB < i1; i += 4 * SN_TB) {   // four independent chains, coalesced loads
        const double a = v[i], b = v[i + SN_TB], c = v[i + 2 * SN_TB], d = v[i + 3 * SN_TB];
        q0 = fma(a, a, q0);
        q1 = fma(b, b, q1);
        q2 = fma(c, c, q2);
        q3 = fma(d, d, q3);
    }
    for (; i < i1; i += SN_TB) {
        const double a = v[i];
        q0 = fma(a, a, q0);
    }
    double q = (q0 + q1) + (q2 + q3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = q;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < SN_TB / 32; ++w) t += red[w];
        parts[blockIdx.x] = t;
        __threadfence();                                   // the partial before the ticket
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();                                       // the ticket before the other partials
    double t = 0.0;
    for (int k = threadIdx.x; k < (int)gridDim.x; k += SN_TB) t += __ldcg(parts + k);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double ss = 0.0;
#pragma unroll
        for (int w = 0; w < SN_TB / 32; ++w) ss += red[w];
        out[0] = sqrt(ss);
    }
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device with that
// device current (every device that loads the library has its own copy of the array).
static int static_scratch_ptr(double** out) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static double* ptr[MAX_DEV];
    static int rc[MAX_DEV];
    static bool done[MAX_DEV];
    int dev = -1;
    GSR_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return GSR_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!done[dev]) {
        int major = 0;
        GSR_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) {
            rc[dev] = GSR_EUNSUPPORTED;   // the library holds sm_100a code only
        } else {
            void* p = nullptr;
            GSR_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
            if (!p) return GSR_ECUDA;
            ptr[dev] = static_cast<double*>(p);
            rc[dev] = GSR_OK;
        }
        done[dev] = true;
    }
    *out = ptr[dev];
    return rc[dev];
}

}  // namespace gsr

using namespace gsr;

extern "C" int gsr_norm2_static(const double* v_dev, int64_t len, double* out_dev, gsr_stream stream) {
    if (!out_dev || len < 0 || (len > 0 && !v_dev)) return GSR_EINVAL;
    if (len > GSR_NORM2_STATIC_MAX_LEN) return GSR_EUNSUPPORTED;   // more partials than the array holds
    double* scratch = nullptr;
    GSR_TRY(static_scratch_ptr(&scratch));
    cudaStream_t s = (cudaStream_t)stream;
    const unsigned grid = len == 0 ? 1u : (unsigned)((len + SN_CHUNK - 1) / SN_CHUNK);
    // the ticket must start at zero, whatever an earlier (possibly failed) call left behind
    GSR_CUDA_TRY(cudaMemsetAsync(scratch, 0, 8, s));
    k_norm2_static<<<grid, SN_TB, 0, s>>>(v_dev, len, scratch, out_dev);
    count_launch();
    GSR_CUDA_TRY(cudaGetLastError());
    return GSR_OK;
}
