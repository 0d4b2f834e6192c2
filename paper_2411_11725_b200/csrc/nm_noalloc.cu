// nm_hext_gradient_noalloc: the uniform-field gradient of nm_llg_adjoint_rhs_hext (Eqs. 31-33)
// for callers that cannot allocate -- no nm_mesh, no workspace, no cudaMalloc / cudaFree, no allocating library call.
//
// The two-pass reduction of nm_local.cu (k_hext_partial / k_hext_final) keeps its per-block partial sums in the
// mesh workspace.  This variant keeps them in a file-scope device array of fixed size instead:
//
//     g_noalloc_part : 3 x NM_NOALLOC_MAX_BLOCKS doubles = 192 KB, resident on every GPU that loads libnm.so
//                      until the process exits; one block sums NM_NOALLOC_BLOCK_NODES = 4096 nodes, which fixes
//                      the largest mesh at NM_NOALLOC_MAX_NODES = 2^25 nodes (256^3 cells has 1.70e7).
//
// Every call on a device shares that array.  A call overwrites the partials it reads (nothing has to start at
// zero, nothing is carried from call to call), so calls that are ordered on the GPU -- same stream, or ordered by
// events -- are independent; calls that OVERLAP on the GPU (different streams, no ordering) race on it and give
// wrong sums.  In host code the array's name is a host-side stand-in, not a device address: the address the
// kernels get is taken with cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>

#include "nm_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kItems = 16;                                   // nodes per thread
constexpr int kBlockNodes = kThreads * kItems;               // 4096
constexpr int kMaxBlocks = (int)(NM_NOALLOC_MAX_NODES / kBlockNodes);   // 8192
static_assert((long long)kMaxBlocks * kBlockNodes == NM_NOALLOC_MAX_NODES, "NM_NOALLOC_MAX_NODES: whole blocks");

static __device__ __align__(256) double g_noalloc_part[3 * kMaxBlocks];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double *g_part_ptr[kMaxDevices];      // device address of g_noalloc_part on device d (null: not asked yet)

// Device address of the scratch array on `device`, which must be current.
nm_status scratch_address(int device, double **out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_part_ptr[device]) {
        double *p = nullptr;
        NM_CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_noalloc_part));
        if (!p) { nm_set_error("cudaGetSymbolAddress gave a null address for the scratch array"); return NM_ECUDA; }
        g_part_ptr[device] = p;
    }
    *out = g_part_ptr[device];
    return NM_OK;
}

__device__ __forceinline__ double block_sum256(double v, double *red)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = l < kThreads / 32 ? red[l] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
    }
    __syncthreads();                  // red is reused by the next call
    return r;                         // valid in thread 0
}

// First pass: part[j * gridDim.x + block] = sum over the block's nodes with (S Ms)_n > 0 of b_n[j],
// b = g' m x a - alpha g' m x (m x a).  Ms = null: every node counts (uniform Ms > 0).
template <typename T>
__global__ void __launch_bounds__(kThreads) k_noalloc_partial(const T *__restrict__ m, const T *__restrict__ av,
                                                              const T *__restrict__ Ms, int N1, int N2, int N3,
                                                              T gp, T agp, double *__restrict__ part)
{
    __shared__ double red[32];
    const int n1 = N1 + 1, n2 = N2 + 1;
    const long long nn = (long long)n1 * n2 * (N3 + 1);
    double s[3] = {0.0, 0.0, 0.0};
#pragma unroll 4
    for (int it = 0; it < kItems; ++it) {
        const long long n = (long long)blockIdx.x * kBlockNodes + it * kThreads + threadIdx.x;
        if (n >= nn) break;
        if (Ms) {       // (S Ms)_n > 0: some cell that contains the node is magnetic
            const int i1 = (int)(n % n1), i2 = (int)((n / n1) % n2), i3 = (int)(n / ((long long)n1 * n2));
            bool inside = false;
            for (int c3 = max(i3 - 1, 0); c3 <= min(i3, N3 - 1); ++c3)
                for (int c2 = max(i2 - 1, 0); c2 <= min(i2, N2 - 1); ++c2)
                    for (int c1 = max(i1 - 1, 0); c1 <= min(i1, N1 - 1); ++c1)
                        inside = inside || Ms[((long long)c3 * N2 + c2) * N1 + c1] > (T)0;
            if (!inside) continue;
        }
        const T mc[3] = {m[n], m[nn + n], m[2 * nn + n]};
        const T ac[3] = {av[n], av[nn + n], av[2 * nn + n]};
        const T mxa[3] = {mc[1] * ac[2] - mc[2] * ac[1], mc[2] * ac[0] - mc[0] * ac[2], mc[0] * ac[1] - mc[1] * ac[0]};
        const T mm[3] = {mc[1] * mxa[2] - mc[2] * mxa[1], mc[2] * mxa[0] - mc[0] * mxa[2], mc[0] * mxa[1] - mc[1] * mxa[0]};
#pragma unroll
        for (int j = 0; j < 3; ++j) s[j] += (double)(gp * mxa[j] - agp * mm[j]);
    }
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double r = block_sum256(s[j], red);
        if (threadIdx.x == 0) part[j * gridDim.x + blockIdx.x] = r;
    }
}

// Second pass: out[j] = -(sum of the block sums), in a fixed order.
__global__ void __launch_bounds__(kThreads) k_noalloc_final(const double *__restrict__ part, int nblocks,
                                                            double *__restrict__ out)
{
    __shared__ double red[32];
    for (int j = 0; j < 3; ++j) {
        double v = 0.0;
        for (int i = threadIdx.x; i < nblocks; i += kThreads) v += part[j * nblocks + i];
        const double r = block_sum256(v, red);
        if (threadIdx.x == 0) out[j] = -r;
    }
}

} // namespace

extern "C" nm_status nm_hext_gradient_noalloc(int device, nm_dtype dtype, const int *n_cells, const void *m,
                                              const void *a, const void *Ms, double gamma, double alpha,
                                              double *dudt_h_out, void *stream)
{
    if (!n_cells || !m || !a || !dudt_h_out) { nm_set_error("nm_hext_gradient_noalloc: NULL argument"); return NM_EINVAL; }
    if (dtype != NM_F32 && dtype != NM_F64) { nm_set_error("nm_hext_gradient_noalloc: dtype %d", (int)dtype); return NM_EINVAL; }
    if (device < 0 || device >= kMaxDevices) {
        nm_set_error("nm_hext_gradient_noalloc: device %d outside 0..%d", device, kMaxDevices - 1);
        return NM_EINVAL;
    }
    const int N1 = n_cells[0], N2 = n_cells[1], N3 = n_cells[2];
    if (N1 < 1 || N2 < 1 || N3 < 1) {
        nm_set_error("nm_hext_gradient_noalloc: n_cells = (%d, %d, %d), every extent must be >= 1", N1, N2, N3);
        return NM_EINVAL;
    }
    const double nodes = ((double)N1 + 1.0) * ((double)N2 + 1.0) * ((double)N3 + 1.0);
    if (nodes > (double)NM_NOALLOC_MAX_NODES) {
        nm_set_error("nm_hext_gradient_noalloc: %.0f nodes exceed NM_NOALLOC_MAX_NODES = %lld (the fixed scratch array "
                     "holds one partial sum per %d nodes); use nm_llg_adjoint_rhs_hext with a mesh workspace",
                     nodes, (long long)NM_NOALLOC_MAX_NODES, kBlockNodes);
        return NM_EINVAL;
    }
    NM_CUDA_TRY(cudaSetDevice(device));
    double *part = nullptr;
    NM_TRY(scratch_address(device, &part));
    const long long nn = (long long)nodes;
    const int nb = (int)((nn + kBlockNodes - 1) / kBlockNodes);
    const double gp = gamma / (1.0 + alpha * alpha);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == NM_F64)
        k_noalloc_partial<double><<<nb, kThreads, 0, st>>>((const double *)m, (const double *)a, (const double *)Ms, N1, N2,
                                                           N3, gp, alpha * gp, part);
    else
        k_noalloc_partial<float><<<nb, kThreads, 0, st>>>((const float *)m, (const float *)a, (const float *)Ms, N1, N2, N3,
                                                          (float)gp, (float)(alpha * gp), part);
    k_noalloc_final<<<1, kThreads, 0, st>>>(part, nb, dudt_h_out);
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}
