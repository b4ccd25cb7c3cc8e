// tdse_observables_noalloc: norm, dipole and dipole acceleration of a device-resident state (row a6; Eq. 34,
// P:302 Eq. 36) for callers that may not allocate: code under CUDA-graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  It is the two-stage reduction of obs_kernel (tdse_kernels.cuh) with its scratch -- per-CTA partial
// sums and the per-member ticket counters -- in a file-scope device array of a fixed size instead of handle-owned
// buffers.  No handle, no cudaMalloc / cudaFree, no allocating library call; the caller passes inputs and outputs.
//
// Every call on a device shares the one array: calls that overlap on the GPU (two streams, two host threads) race on it.
// The array keeps the last call's contents; the counters are cleared in stream order before every launch.
#include <cuda_runtime.h>

#include <mutex>

#include "tdse_device.cuh"

namespace tdse {
namespace {

constexpr int kNaMaxBatch = TDSE_NOALLOC_MAX_BATCH;         // members
constexpr int kNaMaxCtas = TDSE_NOALLOC_MAX_CTAS;           // CTAs of one launch (partial sums: 3 doubles each)
constexpr int kNaRows = 8;                                  // partial waves a thread loads at once
constexpr size_t kNaCounterBytes = sizeof(unsigned int) * kNaMaxBatch;
constexpr size_t kNaScratchBytes = kNaCounterBytes + sizeof(double) * 3 * kNaMaxCtas;      // 16 KiB + 768 KiB

// [counters: kNaMaxBatch x u32][partials: kNaMaxCtas x 3 x f64].  Every GPU that loads the library holds it until exit.
// In HOST code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) unsigned char na_scratch[kNaScratchBytes];

// grid = (ceil(n_r / 256), batch, l segments of rows_per rows).  A thread takes one radial column of its segment; the
// last CTA of a member to sign off adds the member's partials in a fixed order and writes {norm, <z>, <z''>}.
__global__ void __launch_bounds__(256) obs_noalloc_kernel(const double2 *psi, int n_r, int n_l, int batch, double dr,
                                                          double z_nuc, const double *e_now, int rows_per,
                                                          unsigned int *counters, double *partials, double *out) {
    __shared__ double red_s[3 * 8];
    __shared__ int last_flag;
    const int chunks_r = gridDim.x, chunks_l = gridDim.z;
    const int b = blockIdx.y, j = blockIdx.x * 256 + threadIdx.x;
    double red[3] = {0.0, 0.0, 0.0};
    const int l_lo = blockIdx.z * rows_per, l_hi = min(n_l, l_lo + rows_per);
    if (j < n_r) {
        double nn = 0.0, sz = 0.0;
        for (int l0 = l_lo; l0 < l_hi; l0 += kNaRows) {
            const double2 *p = psi + ((size_t)b * n_l + l0) * n_r + j;
            double2 v[kNaRows + 1];
#pragma unroll
            for (int r = 0; r <= kNaRows; ++r) v[r] = (l0 + r < n_l) ? p[(size_t)r * n_r] : make_double2(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < kNaRows; ++r) {
                if (l0 + r >= l_hi) break;
                nn += v[r].x * v[r].x + v[r].y * v[r].y;
                if (l0 + r + 1 < n_l) {
                    const double l = (double)(l0 + r);
                    const double cl = (l + 1.0) / sqrt((2.0 * l + 1.0) * (2.0 * l + 3.0));     // P:94 Eq. 9, m = 0
                    sz = fma(cl, v[r].x * v[r + 1].x + v[r].y * v[r + 1].y, sz);
                }
            }
        }
        const double r = dr * (double)(j + 1);
        red[0] = nn; red[1] = r * sz; red[2] = sz / (r * r);
    }
    block_reduce<256, 3>(red, red_s);
    const int chunks = chunks_r * chunks_l;
    if (threadIdx.x == 0) {
        double *o = partials + ((size_t)b * chunks + blockIdx.x * chunks_l + blockIdx.z) * 3;
        o[0] = red[0]; o[1] = red[1]; o[2] = red[2];
        __threadfence();
        const unsigned int ticket = atomicAdd(counters + b, 1u);
        last_flag = (ticket == (unsigned int)(chunks - 1));
    }
    __syncthreads();
    if (!last_flag) return;
    __threadfence();
    double sum[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < chunks; i += 256) {
        const double *p = partials + ((size_t)b * chunks + i) * 3;
        sum[0] += __ldcg(p); sum[1] += __ldcg(p + 1); sum[2] += __ldcg(p + 2);
    }
    block_reduce<256, 3>(sum, red_s);
    if (threadIdx.x == 0) {
        double *o = out + (size_t)b * 3;
        o[0] = dr * sum[0];
        o[1] = 2.0 * dr * sum[1];
        o[2] = -(e_now ? e_now[b] : 0.0) - 2.0 * z_nuc * dr * sum[2];
        counters[b] = 0u;
    }
}

// Device address of the scratch array, looked up once per device with that device current.
int scratch_address(unsigned char **out) {
    static std::mutex mu;
    static unsigned char *addr[64] = {nullptr};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return TDSE_ERR_CUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned char *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, na_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return TDSE_ERR_CUDA;
        }
        addr[dev] = p;
    }
    *out = addr[dev];
    return TDSE_OK;
}

}  // namespace
}  // namespace tdse

extern "C" int tdse_observables_noalloc(const void *psi_dev, int n_r, int n_l, int batch, double dr, double z_nuc,
                                        const double *e_now_dev, double *out_dev, void *stream) {
    using namespace tdse;
    if (!psi_dev || !out_dev || n_r < 1 || n_l < 1 || batch < 1 || !(dr > 0.0)) return TDSE_ERR_ARG;
    if (batch > kNaMaxBatch) return TDSE_ERR_TOO_LARGE;
    const int chunks_r = (n_r + 255) / 256;
    // l segments: whole multiples of kNaRows rows, about two CTAs per SM when the batch is small
    const long ctas_r = (long)chunks_r * batch;
    const int groups = (n_l + kNaRows - 1) / kNaRows;
    int seg = (int)((2L * 148 + ctas_r - 1) / ctas_r);
    if (seg < 1) seg = 1;
    if (seg > groups) seg = groups;
    const int rows_per = ((groups + seg - 1) / seg) * kNaRows;
    const int chunks_l = (n_l + rows_per - 1) / rows_per;
    if (ctas_r * chunks_l > kNaMaxCtas || chunks_l > 65535) return TDSE_ERR_TOO_LARGE;
    unsigned char *scratch = nullptr;
    const int rc = scratch_address(&scratch);
    if (rc != TDSE_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned int *counters = reinterpret_cast<unsigned int *>(scratch);
    double *partials = reinterpret_cast<double *>(scratch + kNaCounterBytes);
    // the counters must start at zero whatever an earlier (possibly failed) call left behind
    if (cudaMemsetAsync(counters, 0, sizeof(unsigned int) * batch, s) != cudaSuccess) return TDSE_ERR_CUDA;
    obs_noalloc_kernel<<<dim3((unsigned)chunks_r, (unsigned)batch, (unsigned)chunks_l), 256, 0, s>>>(
        static_cast<const double2 *>(psi_dev), n_r, n_l, batch, dr, z_nuc, e_now_dev, rows_per, counters, partials, out_dev);
    return cudaGetLastError() == cudaSuccess ? TDSE_OK : TDSE_ERR_CUDA;
}
