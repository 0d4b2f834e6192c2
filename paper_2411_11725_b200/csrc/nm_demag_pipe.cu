// Pipelined (persistent, TMA-fed) kernels of the fast demag path for fp32 grids with 256 cells
// along the transformed axis -- a2-a4 of the hot path.
//
// Same mathematics and the same blocked, swizzled spectrum layouts as nm_demag_fast.cu; what
// changes is how a CTA is fed.  One persistent CTA per SM walks a static list of tiles; bulk
// asynchronous copies (cp.async.bulk, mbarrier transaction counts) bring tile n+2 into shared
// memory and drain tile n-1 back to HBM while the eight warps transform tile n, so that the load,
// the arithmetic and the store of different tiles overlap on an SM that holds only eight warps
// (the z pass keeps 3 x 16 complex spectrum values plus twiddles per thread: ~250 registers).
//
//   k_pz_mid : z forward, H^ = -N^ M^, z inverse, in place on B[ktl][ky][comp][c3][8].
//              Work item = one folded tensor row |ky| of one k1 tile: the tiles +ky and -ky share
//              the tensor rows, which each warp stages privately (its own k1 column: 6 rows of
//              N3+1 reals) with its own transaction barrier, one item ahead.
#include "nm_async.cuh"
#include "nm_fft16.cuh"
#include "nm_internal.h"

using namespace nmf;
using namespace nma;

namespace {

constexpr int kPipeThreads = 256;

// ---- z pass ------------------------------------------------------------------------------------
struct PzSmem {
    static constexpr int N = 256;
    static constexpr int TILE_ELEMS = 3 * N * TW;                   // complex
    static constexpr int TILE_BYTES = TILE_ELEMS * 8;               // 49152
    static constexpr int NBUF = 3;
    static constexpr int KZP = 258;                                 // tensor |kz| pitch (reals), even
    static constexpr int TSLICE = 6 * KZP;                          // reals per warp (6192 B, one bulk copy)
    static constexpr int WSCR = 2 * Team<16>::SCRATCH - 8;          // scratch per warp: teams at 0 and SCRATCH
    static constexpr int OFF_T = NBUF * TILE_BYTES;
    static constexpr int OFF_SCR = OFF_T + 8 * TSLICE * 4;
    static constexpr int OFF_BAR = OFF_SCR + 8 * WSCR * 8;
    static constexpr int BYTES = OFF_BAR + (NBUF + 8) * 8;
};
static_assert(PzSmem::BYTES <= 227 * 1024, "k_pz_mid shared memory exceeds the sm_100a per-CTA limit");

__global__ void __launch_bounds__(kPipeThreads, 1)
k_pz_mid(float2 *__restrict__ B, const float *__restrict__ Tn, int N2, int nItems, int kt0,
         const float2 *__restrict__ wP)
{
    typedef float T;
    typedef float2 V;
    typedef PzSmem S;
    constexpr int M = 16, N = 256, P = 512;
    extern __shared__ __align__(128) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    T *s_T = reinterpret_cast<T *>(smem + S::OFF_T);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *fullT = fullB + S::NBUF;

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, j = lane >> 1;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    if (tid == 0) {
        for (int q = 0; q < S::NBUF + 8; ++q) mbar_init(fullB + q, 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto tile_ptr = [&](int g, int sub) -> V * {
        const int kyf = g % K2, ktl = g / K2;
        const int ky = sub ? P2 - kyf : kyf;
        return B + ((long long)ktl * P2 + ky) * S::TILE_ELEMS;
    };
    auto n_tiles = [&](int g) -> int {
        const int kyf = g % K2;
        return (kyf == 0 || kyf == N2) ? 1 : 2;
    };
    // this warp's tensor rows of item g: Tn[kt][|ky|][k1 = w][6][KZP], contiguous
    auto load_tensor = [&](int g) {
        const int kyf = g % K2, kt = kt0 + g / K2;
        const T *src = Tn + (((long long)kt * K2 + kyf) * TW + w) * S::TSLICE;
        mbar_expect_tx(fullT + w, S::TSLICE * 4);
        bulk_load(s_T + w * S::TSLICE, src, S::TSLICE * 4, fullT + w);
    };

    // prefetch iterator of thread 0: two tiles ahead of the compute iterator
    int pg = blockIdx.x, psub = 0;
    if (tid == 0) {
        for (int q = 0; q < 2; ++q) {
            if (pg < nItems) {
                mbar_expect_tx(fullB + q, S::TILE_BYTES);
                bulk_load(s_B + q * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + q);
                if (psub + 1 < n_tiles(pg)) ++psub;
                else { pg += G; psub = 0; }
            }
        }
    }
    if (lane == 0 && (int)blockIdx.x < nItems) load_tensor(blockIdx.x);

    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + w * S::WSCR + h * Team<M>::SCRATCH;
    const T *ts = s_T + w * S::TSLICE;
    const int cwj = w ^ swz(j);          // swz(j + 16 t) = swz(j)
    int n = 0;
    uint32_t tphase = 0;

    for (int g = blockIdx.x; g < nItems; g += G) {
        const int kyf = g % K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        for (int sub = 0; sub < nt; ++sub, ++n) {
            const int b = n % S::NBUF;
            mbar_wait(fullB + b, (uint32_t)((n / S::NBUF) & 1));
            V *col = s_B + b * S::TILE_ELEMS + j * TW + cwj;      // element (c, e = j + 16 t): + (c N + 16 t) TW
            V a[3][16];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) a[c][t] = col[(c * N + M * t) * TW];
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) fft_fwd<T, M, true>(a[c], tw, scr, j);
            // H^ = -N^ M^ ; rows of the folded tensor: sign -1 per folded odd axis
            if (sub == 0) {
                mbar_wait(fullT + w, tphase);
                tphase ^= 1;
            }
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                const int kz = 2 * slot_freq<M>(j, s) + h;
                const int kzf = kz <= N ? kz : P - kz;
                const T sz = kz <= N ? (T)1 : (T)-1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                a[0][s] = mk<T>(-(nxx * mx.x + nxy * my_.x + nxz * mz.x), -(nxx * mx.y + nxy * my_.y + nxz * mz.y));
                a[1][s] = mk<T>(-(nxy * mx.x + nyy * my_.x + nyz * mz.x), -(nxy * mx.y + nyy * my_.y + nyz * mz.y));
                a[2][s] = mk<T>(-(nxz * mx.x + nyz * my_.x + nzz * mz.x), -(nxz * mx.y + nyz * my_.y + nzz * mz.y));
            }
            if (sub == nt - 1) {
                __syncwarp();
                if (lane == 0 && g + G < nItems) load_tensor(g + G);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) fft_inv<T, M, true>(a[c], tw, scr, j);
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    V v = a[c][t];
                    v.x += __shfl_xor_sync(0xffffffffu, v.x, 1);
                    v.y += __shfl_xor_sync(0xffffffffu, v.y, 1);
                    if ((t >> 3) == h) col[(c * N + M * t) * TW] = v;
                }
            }
            fence_async_smem();
            __syncthreads();
            if (tid == 0) {
                bulk_store(tile_ptr(g, sub), s_B + b * S::TILE_ELEMS, S::TILE_BYTES);
                bulk_commit();
                bulk_wait_read<1>();          // the store of tile n-1 has left its buffer
                if (pg < nItems) {
                    const int nb = (n + 2) % S::NBUF;
                    mbar_expect_tx(fullB + nb, S::TILE_BYTES);
                    bulk_load(s_B + nb * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + nb);
                    if (psub + 1 < n_tiles(pg)) ++psub;
                    else { pg += G; psub = 0; }
                }
            }
        }
    }
    if (tid == 0) bulk_wait<0>();
}

} // namespace

// ---- host side ----------------------------------------------------------------------------------
bool nm_pipe_mid_ok(const nm_mesh *mesh)
{
    return mesh->fast.on && !mesh->f64 && mesh->fast.M3 == 16 && mesh->fast.Kzp == PzSmem::KZP && mesh->fast.pipe;
}

nm_status nm_pipe_mid(nm_mesh *mesh, int kt0, int nkt, cudaStream_t st)
{
    const NmGeom &g = mesh->g;
    NM_CUDA_TRY(cudaFuncSetAttribute(k_pz_mid, cudaFuncAttributeMaxDynamicSharedMemorySize, PzSmem::BYTES));
    const int nItems = nkt * (g.N2 + 1);
    const int grid = nItems < mesh->sm_count ? nItems : mesh->sm_count;
    NmLaunchScope sc(mesh, NM_K_MID, st);
    k_pz_mid<<<grid, kPipeThreads, PzSmem::BYTES, st>>>((float2 *)mesh->bufB, (const float *)mesh->fast.Tn, g.N2,
                                                        nItems, kt0, (const float2 *)mesh->tw_z);
    return NM_OK;
}
