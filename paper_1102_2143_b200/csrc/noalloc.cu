// noalloc.cu -- msolve_spmv_csr_noalloc: y = A x with the fused <x, A x> of Alg. 1 l.18-19 for
// callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  It needs no handle (msolve_create_* allocates) and calls no cudaMalloc / cudaFree or allocating
// library routine: the only scratch of the operation, one (re, im) partial of the dot product per CTA, lives in a
// file-scope __device__ array of fixed size, which every GPU that loads the library holds until the process exits:
//   MSOLVE_NOALLOC_MAX_ROWS = 2^20 rows / 64 rows per CTA = 16384 CTAs x 2 doubles = 256 KiB.
// It is a variant of k_spmv_csr_vector (spmv.cuh): four lanes per row, rows of a CTA consecutive, per-CTA partials
// written to scratch and summed in a fixed order by a one-CTA kernel (bit-reproducible for given inputs).
//
// The array's name is a host-side stand-in in host code, not a device address; set-up (first call on a device, with
// that device current) asks cudaGetSymbolAddress for the address and the kernels get THAT pointer.
// Every call shares the array and finds the previous call's partials in it.  Nothing in it has to start at zero:
// the reducing kernel reads exactly the gridDim.x partials the SpMV kernel of the same call has written before it
// (same stream), never an entry of an earlier call.  Calls that overlap on the GPU (different streams, or graph
// branches without a dependency) write the same entries and RACE: serialise them.
#include <mutex>

#include "handle.h"
#include "common.cuh"

namespace msolve {

constexpr int kNoAllocThreads = 256;
constexpr int kNoAllocLanes = 4;                                         // lanes per row
constexpr int kNoAllocRowsPerCta = kNoAllocThreads / kNoAllocLanes;      // 64
constexpr long long kNoAllocMaxRows = MSOLVE_NOALLOC_MAX_ROWS;
constexpr int kNoAllocMaxCtas = (int)((kNoAllocMaxRows + kNoAllocRowsPerCta - 1) / kNoAllocRowsPerCta);
constexpr int kNoAllocMaxDevices = 64;

// per-CTA partials of <x, A x>: [cta][re, im]
static __device__ __align__(256) double g_noalloc_partial[2 * kNoAllocMaxCtas];

// One CTA = 64 consecutive rows, 4 lanes per row (lane l takes the non-zeros l, l + 4, ... of its row; the four
// partial sums are added pairwise by shuffles).  Every thread stays in the kernel to the end: the shuffles and the
// CTA reduction need whole warps.
template <typename E>
__global__ void __launch_bounds__(kNoAllocThreads) k_noalloc_spmv_dot(long long n, const int32_t* __restrict__ rowptr,
                                                                      const int32_t* __restrict__ colidx, const E* __restrict__ val,
                                                                      const E* __restrict__ x, E* __restrict__ y, double* partial) {
    __shared__ double red[2 * 32];
    const long long row = (long long)blockIdx.x * kNoAllocRowsPerCta + threadIdx.x / kNoAllocLanes;
    const int sub = threadIdx.x % kNoAllocLanes;
    const bool valid = row < n;
    int j = 0, e = 0;
    if (valid) { j = rowptr[row] + sub; e = rowptr[row + 1]; }
    E sum = cmake<E>(0.0, 0.0);
    for (; j < e; j += kNoAllocLanes) sum = cfma(ld_stream(val + j), ld_ro(x + colidx[j]), sum);
#pragma unroll
    for (int o = kNoAllocLanes / 2; o > 0; o >>= 1) sum = cshfl_xor_add(sum, o);
    double acc[2] = {0.0, 0.0};
    if (valid && sub == 0) {
        y[row] = sum;
        const E xi = x[row];
        acc[0] = cdot_re(xi, sum);                                       // conj(x_i) y_i
        acc[1] = cdot_im(xi, sum);
    }
    block_sum<2>(acc, red);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = acc[0]; partial[2 * blockIdx.x + 1] = acc[1]; }
}

// dot[0..1] = sum of the first `count` partials, in a fixed order (thread t adds t, t + 256, ...; then the CTA tree)
__global__ void __launch_bounds__(kNoAllocThreads) k_noalloc_reduce(const double* partial, int count, double* dot) {
    __shared__ double red[2 * 32];
    double acc[2] = {0.0, 0.0};
    for (int c = threadIdx.x; c < count; c += kNoAllocThreads) { acc[0] += partial[2 * c]; acc[1] += partial[2 * c + 1]; }
    block_sum<2>(acc, red);
    if (threadIdx.x == 0) { dot[0] = acc[0]; dot[1] = acc[1]; }
}

// set-up, once per device: the device address of the scratch array on the CURRENT device
static int noalloc_scratch(double** out) {
    static std::mutex mu;
    static double* ptr[kNoAllocMaxDevices] = {};
    int dev = -1;
    MSOLVE_CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: device ordinal %d not supported (< %d)", dev, kNoAllocMaxDevices);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        MSOLVE_CU(cudaGetSymbolAddress(&p, g_noalloc_partial));
        if (!p) return fail(MSOLVE_ECUDA, "msolve_spmv_csr_noalloc: cudaGetSymbolAddress returned NULL");
        ptr[dev] = (double*)p;
    }
    *out = ptr[dev];
    return MSOLVE_OK;
}

template <typename E>
static int noalloc_launch(long long n, const int32_t* rowptr, const int32_t* colidx, const void* val, const void* x, void* y,
                          double* dot, double* scratch, cudaStream_t s) {
    const int grid = (int)((n + kNoAllocRowsPerCta - 1) / kNoAllocRowsPerCta);
    if (grid > 0) {
        k_noalloc_spmv_dot<E><<<grid, kNoAllocThreads, 0, s>>>(n, rowptr, colidx, (const E*)val, (const E*)x, (E*)y, scratch);
        MSOLVE_CU(cudaGetLastError());
    }
    k_noalloc_reduce<<<1, kNoAllocThreads, 0, s>>>(scratch, grid, dot);
    MSOLVE_CU(cudaGetLastError());
    return MSOLVE_OK;
}

}  // namespace msolve

using namespace msolve;

extern "C" int msolve_spmv_csr_noalloc(int64_t n, const int32_t* d_rowptr, const int32_t* d_colidx, const void* d_val, int dtype,
                                       const void* d_x, void* d_y, double* d_dot, void* stream) {
    if (dtype != MSOLVE_C64 && dtype != MSOLVE_C128 && dtype != MSOLVE_F32 && dtype != MSOLVE_F64)
        return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: unknown dtype %d", dtype);
    if (n < 0) return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: n < 0");
    if (n > kNoAllocMaxRows)
        return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: n = %lld exceeds MSOLVE_NOALLOC_MAX_ROWS = %lld (the scratch array is static; "
                    "larger systems go through msolve_create_csr + msolve_spmv)", (long long)n, kNoAllocMaxRows);
    if (!d_dot || !d_rowptr) return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: d_rowptr / d_dot is NULL");
    if (n > 0 && (!d_x || !d_y)) return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: d_x / d_y is NULL");
    const size_t eb = elem_bytes(dtype);
    if (((uintptr_t)d_val % eb) || ((uintptr_t)d_x % eb) || ((uintptr_t)d_y % eb) || ((uintptr_t)d_dot % 8u) ||
        ((uintptr_t)d_rowptr % 4u) || ((uintptr_t)d_colidx % 4u))
        return fail(MSOLVE_EINVAL, "msolve_spmv_csr_noalloc: a pointer is not aligned to its element size");
    double* scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc != MSOLVE_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    switch (dtype) {
        case MSOLVE_C128: return noalloc_launch<double2>(n, d_rowptr, d_colidx, d_val, d_x, d_y, d_dot, scratch, s);
        case MSOLVE_C64:  return noalloc_launch<float2>(n, d_rowptr, d_colidx, d_val, d_x, d_y, d_dot, scratch, s);
        case MSOLVE_F64:  return noalloc_launch<double>(n, d_rowptr, d_colidx, d_val, d_x, d_y, d_dot, scratch, s);
        default:          return noalloc_launch<float>(n, d_rowptr, d_colidx, d_val, d_x, d_y, d_dot, scratch, s);
    }
}
