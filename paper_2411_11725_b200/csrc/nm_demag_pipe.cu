// Pipelined (persistent, TMA-fed) kernels of the fast demag path for fp32 grids with 256 cells
// along the transformed axis -- a2-a4 of the hot path.
//
// Same mathematics and the same blocked, swizzled spectrum layouts as nm_demag_fast.cu; what
// changes is how a CTA is fed.  One persistent CTA per SM walks a static list of tiles; bulk
// asynchronous copies (cp.async.bulk, mbarrier transaction counts) bring tile n+2 into shared
// memory and drain tile n-1 back to HBM while the eight warps transform tile n, so that the load,
// the arithmetic and the store of different tiles overlap on an SM that holds only eight warps
// (the z pass keeps 3 x 16 complex spectrum values plus twiddles per thread).  In the z pass a
// ninth warp issues the copies and the transform warps synchronise only through the tile
// barriers (full / done), never with one another.
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
    static constexpr int BYTES = OFF_BAR + (2 * NBUF + 8) * 8;
};
constexpr int kMidThreads = 288;      // eight transform warps and one copy warp
static_assert(PzSmem::BYTES <= 227 * 1024, "k_pz_mid shared memory exceeds the sm_100a per-CTA limit");

// EMB: the mesh has n3v < 256 cell layers (embedded, nm_fast_plan): rows c3 >= n3v of a tile were
// never written and enter the transform as zeros.
template <bool EMB>
__global__ void __launch_bounds__(kMidThreads, 1)
k_pz_mid(float2 *__restrict__ B, const float *__restrict__ Tn, int N2, int nItems, int kt0,
         const float2 *__restrict__ wP, int n3v)
{
    typedef float T;
    typedef float2 V;
    typedef PzSmem S;
    constexpr int M = 16, N = 256, P = 512;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    T *s_T = reinterpret_cast<T *>(smem + S::OFF_T);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *doneB = fullB + S::NBUF;
    uint64_t *fullT = doneB + S::NBUF;

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, j = lane >> 1;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    if (tid == 0) {
        for (int q = 0; q < S::NBUF; ++q) {
            mbar_init(fullB + q, 1);
            mbar_init(doneB + q, 8);
        }
        for (int q = 0; q < 8; ++q) mbar_init(fullT + q, 1);
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

    // ---- copy warp: one thread walks the same tile list; it stores tile n as soon as the eight
    // transform warps have left it and refills the buffer with tile n + NBUF at once, so the transform
    // warps never wait for one another and drift into different phases (butterflies of one warp
    // over the scratch exchange of another)
    if (w == 8) {
        if (lane != 0) return;
        int pg = blockIdx.x, psub = 0;
        for (int q = 0; q < S::NBUF; ++q) {
            if (pg < nItems) {
                mbar_expect_tx(fullB + q, S::TILE_BYTES);
                bulk_load(s_B + q * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + q);
                if (psub + 1 < n_tiles(pg)) ++psub;
                else { pg += G; psub = 0; }
            }
        }
        int n = 0;
        for (int g = blockIdx.x; g < nItems; g += G) {
            const int nt = n_tiles(g);
            for (int sub = 0; sub < nt; ++sub, ++n) {
                const int b = n % S::NBUF;
                mbar_wait_idle(doneB + b, (uint32_t)((n / S::NBUF) & 1));
                bulk_store(tile_ptr(g, sub), s_B + b * S::TILE_ELEMS, S::TILE_BYTES);
                bulk_commit();
                bulk_wait_read<0>();          // the store has left the buffer: refill it with tile n + NBUF
                if (pg < nItems) {
                    mbar_expect_tx(fullB + b, S::TILE_BYTES);
                    bulk_load(s_B + b * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + b);
                    if (psub + 1 < n_tiles(pg)) ++psub;
                    else { pg += G; psub = 0; }
                }
            }
        }
        bulk_wait<0>();
        return;
    }
    if (lane == 0 && (int)blockIdx.x < nItems) load_tensor(blockIdx.x);

    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + w * S::WSCR + h * Team<M>::SCRATCH;
    const T *ts = s_T + w * S::TSLICE;
    const int cw0 = w ^ swz(j);          // swz(j + 16 t) = swz(j)
    int n = 0;
    uint32_t tphase = 0;

    for (int g = blockIdx.x; g < nItems; g += G) {
        const int kyf = g % K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        for (int sub = 0; sub < nt; ++sub, ++n) {
            const int b = n % S::NBUF;
            mbar_wait(fullB + b, (uint32_t)((n / S::NBUF) & 1));
            const int cwj = cw0 ^ swz(sub ? P2 - kyf : kyf);     // rows of B are swizzled by c3 and by ky
            V *col = s_B + b * S::TILE_ELEMS + j * TW + cwj;      // element (c, e = j + 16 t): + (c N + 16 t) TW
            V a[3][16];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    a[c][t] = col[(c * N + M * t) * TW];
                    if (EMB && j + M * t >= n3v) a[c][t] = mk<T>((T)0, (T)0);
                }
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
            // three forward transforms, the butterflies of one component between the scratch
            // stores and loads of another (one scratch per team: put(c + 1) follows get(c))
            dft16<T, false>(a[0]);
            fwd_put<T, M, true>(a[0], tw, scr, j);
            dft16<T, false>(a[1]);
            fwd_get<T, M>(a[0], scr, j);
            dft16<T, false>(a[2]);
            fwd_put<T, M, true>(a[1], tw, scr, j);
            dft16<T, false>(a[0]);
            fwd_get<T, M>(a[1], scr, j);
            fwd_put<T, M, true>(a[2], tw, scr, j);
            dft16<T, false>(a[1]);
            fwd_get<T, M>(a[2], scr, j);
            dft16<T, false>(a[2]);
            // H^ = -N^ M^ ; rows of the folded tensor: sign -1 per folded odd axis
            if (sub == 0) {
                mbar_wait(fullT + w, tphase);
                tphase ^= 1;
            }
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                // kz = 2 j + 32 rev16(s) + h: which side of the fold it lies on is fixed by the slot,
                // except for the slot that straddles kz = N
                const int rs = rev16(s);
                const int kz = 2 * slot_freq<M>(j, s) + h;
                const bool up = rs > 8 || (rs == 8 && (j | h) != 0);
                const int kzf = up ? P - kz : kz;
                const T sz = up ? (T)-1 : (T)1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
                const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
                const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
                a[0][s] = mk<T>(-hx.x, -hx.y);
                a[1][s] = mk<T>(-hy.x, -hy.y);
                a[2][s] = mk<T>(-hz.x, -hz.y);
            }
            if (sub == nt - 1) {
                __syncwarp();
                if (lane == 0 && g + G < nItems) load_tensor(g + G);
            }
            dft16<T, true>(a[0]);
            inv_put<T, M>(a[0], scr, j);
            dft16<T, true>(a[1]);
            inv_get<T, M, true>(a[0], tw, scr, j);
            dft16<T, true>(a[2]);
            inv_put<T, M>(a[1], scr, j);
            dft16<T, true>(a[0]);
            inv_get<T, M, true>(a[1], tw, scr, j);
            inv_put<T, M>(a[2], scr, j);
            dft16<T, true>(a[1]);
            inv_get<T, M, true>(a[2], tw, scr, j);
            dft16<T, true>(a[2]);
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
            // even + odd half: the lane of half h keeps rows t = s + 8 h (half_sum)
            V *colh = col + (size_t)h * 8 * M * TW;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int s = 0; s < 8; ++s) colh[(c * N + M * s) * TW] = half_sum(a[c], s, h);
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(doneB + b);
        }
    }
}


// ---- z pass, 192 cells along z -----------------------------------------------------------------------
// k_pz_mid for N3 = 192 = 3 x 64 (Len<12>, nm_fft16.cuh): the same pipeline (copy warp, three-deep tile ring,
// per-warp tensor slices); a warp still owns one k1 column, its lanes are (l, j, h) = (sub-sequence, thread of the
// M = 4 team, half), lanes with l = 3 idle; the radix-3 step sits between the 64-point transforms and the tensor
// product, two lane exchanges per slot.
struct Pz3Smem {
    static constexpr int N = 192;
    static constexpr int TILE_ELEMS = 3 * N * TW;                   // complex
    static constexpr int TILE_BYTES = TILE_ELEMS * 8;               // 36864
    static constexpr int NBUF = 4;
    static constexpr int KZP = 194;                                 // tensor |kz| pitch (reals), even
    static constexpr int TSLICE = 6 * KZP;                          // reals per warp (4656 B, one bulk copy)
    static constexpr int WSCR = 2 * Team<4>::SCRATCH - 8;
    static constexpr int OFF_T = NBUF * TILE_BYTES;
    static constexpr int OFF_SCR = OFF_T + 8 * TSLICE * 4;
    static constexpr int OFF_BAR = OFF_SCR + 8 * WSCR * 8;
    static constexpr int BYTES = OFF_BAR + (2 * NBUF + 8) * 8;
};
static_assert(Pz3Smem::BYTES <= 227 * 1024, "k_pz_mid3 shared memory exceeds the sm_100a per-CTA limit");

template <bool EMB>
__global__ void __launch_bounds__(kMidThreads, 1)
k_pz_mid3(float2 *__restrict__ B, const float *__restrict__ Tn, int N2, int nItems, int kt0,
          const float2 *__restrict__ wP, int n3v)
{
    typedef float T;
    typedef float2 V;
    typedef Pz3Smem S;
    constexpr int MI = 4, N = 192, P = 384;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    T *s_T = reinterpret_cast<T *>(smem + S::OFF_T);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *doneB = fullB + S::NBUF;
    uint64_t *fullT = doneB + S::NBUF;

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, i = lane >> 1, j = i & 3, l = min(i >> 2, 2);
    const bool act = (i >> 2) < 3;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    if (tid == 0) {
        for (int q = 0; q < S::NBUF; ++q) {
            mbar_init(fullB + q, 1);
            mbar_init(doneB + q, 8);
        }
        for (int q = 0; q < 8; ++q) mbar_init(fullT + q, 1);
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
    auto load_tensor = [&](int g) {
        const int kyf = g % K2, kt = kt0 + g / K2;
        const T *src = Tn + (((long long)kt * K2 + kyf) * TW + w) * S::TSLICE;
        mbar_expect_tx(fullT + w, S::TSLICE * 4);
        bulk_load(s_T + w * S::TSLICE, src, S::TSLICE * 4, fullT + w);
    };

    if (w == 8) {           // copy warp, as in k_pz_mid
        if (lane != 0) return;
        int pg = blockIdx.x, psub = 0;
        for (int q = 0; q < S::NBUF; ++q) {
            if (pg < nItems) {
                mbar_expect_tx(fullB + q, S::TILE_BYTES);
                bulk_load(s_B + q * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + q);
                if (psub + 1 < n_tiles(pg)) ++psub;
                else { pg += G; psub = 0; }
            }
        }
        int n = 0;
        for (int g = blockIdx.x; g < nItems; g += G) {
            const int nt = n_tiles(g);
            for (int sub = 0; sub < nt; ++sub, ++n) {
                const int b = n % S::NBUF;
                mbar_wait_idle(doneB + b, (uint32_t)((n / S::NBUF) & 1));
                bulk_store(tile_ptr(g, sub), s_B + b * S::TILE_ELEMS, S::TILE_BYTES);
                bulk_commit();
                bulk_wait_read<0>();
                if (pg < nItems) {
                    mbar_expect_tx(fullB + b, S::TILE_BYTES);
                    bulk_load(s_B + b * S::TILE_ELEMS, tile_ptr(pg, psub), S::TILE_BYTES, fullB + b);
                    if (psub + 1 < n_tiles(pg)) ++psub;
                    else { pg += G; psub = 0; }
                }
            }
        }
        bulk_wait<0>();
        return;
    }
    if (lane == 0 && (int)blockIdx.x < nItems) load_tensor(blockIdx.x);

    // stage twiddles of the 64-point transforms in the TW0 form with the slot-position part of the radix-3 twiddle
    // folded in, w_384^((3 j + l)(2 t' + h)), and the rest of that twiddle, w_12^(l p) (r3_fwd); wP = exp(-2 pi i q / 384)
    V tw[16], tw3[3];
#pragma unroll
    for (int t = 0; t < 16; ++t) tw[t] = wP[(3 * j + l) * (2 * t + h)];
#pragma unroll
    for (int q = 0; q < 3; ++q) tw3[q] = wP[32 * l * (q + 1)];
    V *scr = s_scr + w * S::WSCR + h * Team<MI>::SCRATCH;
    const T *ts = s_T + w * S::TSLICE;
    int n = 0;
    uint32_t tphase = 0;

    for (int g = blockIdx.x; g < nItems; g += G) {
        const int kyf = g % K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        for (int sub = 0; sub < nt; ++sub, ++n) {
            const int b = n % S::NBUF;
            mbar_wait(fullB + b, (uint32_t)((n / S::NBUF) & 1));
            const int cw = w ^ swz(sub ? P2 - kyf : kyf);        // rows of B are swizzled by c3 and by ky
            V *tile = s_B + b * S::TILE_ELEMS;
            V a[3][16];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    const int e = 3 * (j + MI * t) + l;
                    a[c][t] = tile[(c * N + e) * TW + (cw ^ swz(e))];
                    if (EMB && e >= n3v) a[c][t] = mk<T>((T)0, (T)0);
                }
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
            dft16<T, false>(a[0]);
            fwd_put<T, MI, true>(a[0], tw, scr, i);
            dft16<T, false>(a[1]);
            fwd_get<T, MI>(a[0], scr, i);
            dft16<T, false>(a[2]);
            fwd_put<T, MI, true>(a[1], tw, scr, i);
            dftM<T, false, MI>(a[0]);
            fwd_get<T, MI>(a[1], scr, i);
            fwd_put<T, MI, true>(a[2], tw, scr, i);
            dftM<T, false, MI>(a[1]);
            r3_fwd<T>(a[0], tw3, lane, l);
            fwd_get<T, MI>(a[2], scr, i);
            dftM<T, false, MI>(a[2]);
            r3_fwd<T>(a[1], tw3, lane, l);
            r3_fwd<T>(a[2], tw3, lane, l);
            if (sub == 0) {
                mbar_wait(fullT + w, tphase);
                tphase ^= 1;
            }
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                const int kz = 2 * slot_freq<MI>(j, s) + h + 128 * l;
                const bool up = kz > N;
                const int kzf = up ? P - kz : kz;
                const T sz = up ? (T)-1 : (T)1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
                const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
                const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
                a[0][s] = mk<T>(-hx.x, -hx.y);
                a[1][s] = mk<T>(-hy.x, -hy.y);
                a[2][s] = mk<T>(-hz.x, -hz.y);
            }
            if (sub == nt - 1) {
                __syncwarp();
                if (lane == 0 && g + G < nItems) load_tensor(g + G);
            }
            r3_inv<T>(a[0], tw3, lane, l);
            dftM<T, true, MI>(a[0]);
            inv_put<T, MI>(a[0], scr, i);
            r3_inv<T>(a[1], tw3, lane, l);
            dftM<T, true, MI>(a[1]);
            inv_get<T, MI, true>(a[0], tw, scr, i);
            r3_inv<T>(a[2], tw3, lane, l);
            dftM<T, true, MI>(a[2]);
            inv_put<T, MI>(a[1], scr, i);
            dft16<T, true>(a[0]);
            inv_get<T, MI, true>(a[1], tw, scr, i);
            inv_put<T, MI>(a[2], scr, i);
            dft16<T, true>(a[1]);
            inv_get<T, MI, true>(a[2], tw, scr, i);
            dft16<T, true>(a[2]);
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int s = 0; s < 8; ++s) {
                    const int e = 3 * (j + MI * (s + 8 * h)) + l;
                    const V v = half_sum(a[c], s, h);
                    if (act) tile[(c * N + e) * TW + (cw ^ swz(e))] = v;
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(doneB + b);
        }
    }
}


// ---- z pass, 128 cells along z ---------------------------------------------------------------------
// The same pipeline for N3 = 128 (M = 8): a team transforms two lines at once, so a warp owns two
// columns of a tile and four warps a whole tile; warps 0-3 take the +ky tile of an item and warps
// 4-7 the -ky tile at the same time (both read the same folded tensor rows, staged once per column
// pair).  A buffer holds the tile pair of one item (2 x 24 KB).  The copy warp also brings the
// tensor rows of item n + 1 as soon as the eight warps have finished the products of item n
// (`freeT`), half an item before it stores item n.
struct Pz8Smem {
    static constexpr int N = 128;
    static constexpr int TILE_ELEMS = 3 * N * TW;                   // complex
    static constexpr int TILE_BYTES = TILE_ELEMS * 8;               // 24576
    static constexpr int SLOT_ELEMS = 2 * TILE_ELEMS;
    static constexpr int NBUF = 3;
    static constexpr int KZP = 130;                                 // tensor |kz| pitch (reals), even
    static constexpr int TSLICE = 2 * 6 * KZP;                      // reals per column pair (6240 B, one bulk copy)
    static constexpr int WSCR = 2 * Team<8>::SCRATCH - 8;
    static constexpr int OFF_T = NBUF * 2 * TILE_BYTES;
    static constexpr int OFF_SCR = OFF_T + 4 * TSLICE * 4;
    static constexpr int OFF_BAR = OFF_SCR + 8 * WSCR * 8;
    static constexpr int BYTES = OFF_BAR + (2 * NBUF + 2) * 8;
};
static_assert(Pz8Smem::BYTES <= 227 * 1024, "k_pz_mid8 shared memory exceeds the sm_100a per-CTA limit");
static_assert((Pz8Smem::TSLICE * 4) % 16 == 0 && Pz8Smem::OFF_SCR % 16 == 0 && Pz8Smem::OFF_BAR % 8 == 0, "alignment");

template <bool EMB>
__global__ void __launch_bounds__(kMidThreads, 1)
k_pz_mid8(float2 *__restrict__ B, const float *__restrict__ Tn, int N2, int nItems, int kt0,
          const float2 *__restrict__ wP, int n3v)
{
    typedef float T;
    typedef float2 V;
    typedef Pz8Smem S;
    constexpr int M = 8, N = 128, P = 256;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    T *s_T = reinterpret_cast<T *>(smem + S::OFF_T);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *doneB = fullB + S::NBUF;
    uint64_t *fullT = doneB + S::NBUF;      // one barrier for the four slices of an item
    uint64_t *freeT = fullT + 1;

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    if (tid == 0) {
        for (int q = 0; q < S::NBUF; ++q) {
            mbar_init(fullB + q, 1);
            mbar_init(doneB + q, 8);
        }
        mbar_init(fullT, 1);
        mbar_init(freeT, 8);
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

    if (w == 8) {           // copy warp
        if (lane != 0) return;
        auto load_item = [&](int g, int b) {
            const int nt = n_tiles(g);
            mbar_expect_tx(fullB + b, nt * S::TILE_BYTES);
            for (int sub = 0; sub < nt; ++sub)
                bulk_load(s_B + b * S::SLOT_ELEMS + sub * S::TILE_ELEMS, tile_ptr(g, sub), S::TILE_BYTES, fullB + b);
        };
        // tensor rows of item g: Tn[kt][|ky|][k1 = 0..7][6][KZP], the eight columns contiguous
        auto load_tensor = [&](int g) {
            const int kyf = g % K2, kt = kt0 + g / K2;
            const T *src = Tn + ((long long)kt * K2 + kyf) * TW * 6 * S::KZP;
            mbar_expect_tx(fullT, 4 * S::TSLICE * 4);
            bulk_load(s_T, src, 4 * S::TSLICE * 4, fullT);
        };
        int pg = blockIdx.x;
        for (int q = 0; q < S::NBUF; ++q, pg += G)
            if (pg < nItems) load_item(pg, q);
        if ((int)blockIdx.x < nItems) load_tensor(blockIdx.x);
        int n = 0;
        for (int g = blockIdx.x; g < nItems; g += G, ++n) {
            const int b = n % S::NBUF;
            mbar_wait_idle(freeT, (uint32_t)(n & 1));       // the products of item n are done
            if (g + G < nItems) load_tensor(g + G);
            mbar_wait_idle(doneB + b, (uint32_t)((n / S::NBUF) & 1));
            const int nt = n_tiles(g);
            for (int sub = 0; sub < nt; ++sub)
                bulk_store(tile_ptr(g, sub), s_B + b * S::SLOT_ELEMS + sub * S::TILE_ELEMS, S::TILE_BYTES);
            bulk_commit();
            bulk_wait_read<0>();
            if (pg < nItems) {
                load_item(pg, b);
                pg += G;
            }
        }
        bulk_wait<0>();
        return;
    }

    // ---- transform warps: warp = (which tile of the pair, column pair), lane = (line, j, half)
    const int sub = w >> 2, cp = w & 3;
    const int h = lane & 1, i = lane >> 1;
    const int l = i >> 3, j = i & 7;
    const int k1 = 2 * cp + l;
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + w * S::WSCR + h * Team<M>::SCRATCH;
    const T *ts = s_T + k1 * 6 * S::KZP;
    int n = 0;
    for (int g = blockIdx.x; g < nItems; g += G, ++n) {
        const int kyf = g % K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        const int b = n % S::NBUF;
        if (sub < nt) {
            mbar_wait(fullB + b, (uint32_t)((n / S::NBUF) & 1));
            // element (c, e = j + 8 t) of column k1: row (c N + e), slot k1 ^ swz(e) ^ swz(ky);
            // swz(j + 8 t) = (j >> 1) ^ 4 (t & 1)
            const int cw = k1 ^ swz(sub ? P2 - kyf : kyf) ^ (j >> 1);
            V *colE = s_B + b * S::SLOT_ELEMS + sub * S::TILE_ELEMS + j * TW + cw;
            V *colO = s_B + b * S::SLOT_ELEMS + sub * S::TILE_ELEMS + j * TW + (cw ^ 4);
            V a[3][16];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    a[c][t] = ((t & 1) ? colO : colE)[(c * N + M * t) * TW];
                    if (EMB && j + M * t >= n3v) a[c][t] = mk<T>((T)0, (T)0);
                }
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) fft_fwd<T, M, true>(a[c], tw, scr, i);
            // H^ = -N^ M^ ; rows of the folded tensor: sign -1 per folded odd axis
            mbar_wait(fullT, (uint32_t)(n & 1));
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                // kz = 2 (2 j + u + 16 rev8(p)) + h, s = 8 u + p: the side of the fold is fixed by the
                // slot, except for the slot that straddles kz = N
                const int u = s / M, r8 = rev8(s % M);
                const int kz = 2 * slot_freq<M>(j, s) + h;
                const bool up = r8 > 4 || (r8 == 4 && (j | u | h) != 0);
                const int kzf = up ? P - kz : kz;
                const T sz = up ? (T)-1 : (T)1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
                const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
                const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
                a[0][s] = mk<T>(-hx.x, -hx.y);
                a[1][s] = mk<T>(-hy.x, -hy.y);
                a[2][s] = mk<T>(-hz.x, -hz.y);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(freeT);
#pragma unroll
            for (int c = 0; c < 3; ++c) fft_inv<T, M, true>(a[c], tw, scr, i);
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int s = 0; s < 8; ++s) ((s & 1) ? colO : colE)[(c * N + M * (s + 8 * h)) * TW] = half_sum(a[c], s, h);
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(doneB + b);
        } else {                    // the item has one tile only: this warp just keeps the barrier counts,
            // after the same waits as a working warp (an arrival must not run into the previous phase)
            mbar_wait(fullB + b, (uint32_t)((n / S::NBUF) & 1));
            mbar_wait(fullT, (uint32_t)(n & 1));
            if (lane == 0) {
                mbar_arrive(freeT);
                mbar_arrive(doneB + b);
            }
        }
    }
}


// ---- z pass, fp64, 256 cells along z ---------------------------------------------------------------
// One shared-memory region serves, in turn, the spectrum tile of a work item (3 x 256 x 8 complex
// doubles, 96 KB) and the folded tensor rows of its eight columns (8 x 6 x 258 doubles, 96.75 KB):
// a warp pulls its column of the tile into registers (3 x 16 complex doubles per thread, which is
// what an fp64 thread can hold -- the stage twiddles live in a shared-memory table); the last warp
// to have done so has the tensor rows copied over the tile while the forward transforms run; the last
// warp to finish its products has the next tile copied over the tensor rows while the inverse
// transforms run.  Results go straight from registers to B (16-byte stores, the eight warps of a CTA
// fill the 128-byte rows between them), so no output tile is staged and both bulk copies have a whole
// transform phase to land.  No CTA-wide barrier inside the loop: warps meet only at the two counters.
struct Pz64Smem {
    static constexpr int N = 256;
    static constexpr int TILE_ELEMS = 3 * N * TW;                   // complex doubles
    static constexpr int TILE_BYTES = TILE_ELEMS * 16;              // 98304
    static constexpr int KZP = 258;                                 // tensor |kz| pitch (reals), even
    static constexpr int TSLICE = 6 * KZP;                          // reals per column
    static constexpr int TENS_BYTES = TW * TSLICE * 8;              // 99072, one bulk copy
    static constexpr int REGION = TENS_BYTES > TILE_BYTES ? TENS_BYTES : TILE_BYTES;
    static constexpr int OFF_SCR = REGION;
    static constexpr int SCR_BYTES = 16 * Team<16>::SCRATCH64 * 16; // 70656
    static constexpr int OFF_TW = OFF_SCR + SCR_BYTES;
    static constexpr int TW_BYTES = 16 * 32 * 16;                   // [t'][lane]
    static constexpr int OFF_BAR = OFF_TW + TW_BYTES;
    static constexpr int BYTES = OFF_BAR + 32;
};
static_assert(Pz64Smem::BYTES <= 227 * 1024, "k_pz_mid64 shared memory exceeds the sm_100a per-CTA limit");
static_assert(Pz64Smem::OFF_SCR % 128 == 0 && Pz64Smem::OFF_TW % 16 == 0 && Pz64Smem::OFF_BAR % 8 == 0, "alignment");

// arrival on a CTA-local counter, ordered after this thread's earlier accesses and before its later
// ones; returns the count before the arrival
__device__ __forceinline__ unsigned arrive_count(unsigned *cnt)
{
    unsigned old;
    asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(cnt)) : "memory");
    return old;
}

template <bool EMB>
__global__ void __launch_bounds__(kPipeThreads, 1)
k_pz_mid64(double2 *__restrict__ B, const double *__restrict__ Tn, int N2, int nItems, int kt0,
           const double2 *__restrict__ wP, int n3v)
{
    typedef double T;
    typedef double2 V;
    typedef Pz64Smem S;
    constexpr int M = 16, N = 256, P = 512;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    const T *s_T = reinterpret_cast<const T *>(smem);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    V *s_tw = reinterpret_cast<V *>(smem + S::OFF_TW);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *fullT = fullB + 1;
    unsigned *cnt = reinterpret_cast<unsigned *>(fullT + 1);        // [0]: columns in registers, [1]: products done

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, j = lane >> 1;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    auto tile_ptr = [&](int g, int sub) -> V * {
        const int kyf = g % K2, ktl = g / K2;
        const int ky = sub ? P2 - kyf : kyf;
        return B + ((long long)ktl * P2 + ky) * S::TILE_ELEMS;
    };
    if (tid == 0) {
        mbar_init(fullB, 1);
        mbar_init(fullT, 1);
        cnt[0] = cnt[1] = 0;
        mbar_fence_init();
    }
    // stage twiddles of every lane: w_P^(j (2 t' + h)) (load_twiddles_h), conflict-free by lane
    for (int q = tid; q < 16 * 32; q += kPipeThreads) {
        const int tp = q >> 5, ln = q & 31;
        s_tw[q] = wP[((ln >> 1) * (2 * tp + (ln & 1))) & (P - 1)];
    }
    __syncthreads();
    if (tid == 0 && (int)blockIdx.x < nItems) {
        mbar_expect_tx(fullB, S::TILE_BYTES);
        bulk_load(s_B, tile_ptr(blockIdx.x, 0), S::TILE_BYTES, fullB);
    }
    const V *tws = s_tw + lane;
    V *scr = s_scr + (2 * w + h) * Team<M>::SCRATCH64;
    const T *ts = s_T + w * S::TSLICE;
    const int cw0 = w ^ swzT<T>(j);      // swz(j + 16 t) = swz(j)
    uint32_t ph = 0;

    for (int g = blockIdx.x; g < nItems; g += G) {
        const int kyf = g % K2, kt = kt0 + g / K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        for (int sub = 0; sub < nt; ++sub, ph ^= 1) {
            mbar_wait(fullB, ph);
            const int cwj = cw0 ^ swzT<T>(sub ? P2 - kyf : kyf); // rows of B are swizzled by c3 and by ky
            const int coff = j * TW + cwj;                        // element (c, e = j + 16 t): + (c N + 16 t) TW
            V a[3][16];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    a[c][t] = s_B[coff + (c * N + M * t) * TW];
                    if (EMB && j + M * t >= n3v) a[c][t] = mk<T>((T)0, (T)0);
                }
            }
            __syncwarp();
            if (lane == 0 && (arrive_count(cnt) & 7) == 7) {     // every column is in registers: bring the tensor rows
                mbar_expect_tx(fullT, S::TENS_BYTES);
                bulk_load(smem, Tn + ((long long)kt * K2 + kyf) * TW * S::TSLICE, S::TENS_BYTES, fullT);
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
            dft16<T, false>(a[0]);
            fwd_put_s<T, M, 32>(a[0], tws, scr, j);
            dft16<T, false>(a[1]);
            fwd_get<T, M>(a[0], scr, j);
            dft16<T, false>(a[2]);
            fwd_put_s<T, M, 32>(a[1], tws, scr, j);
            dft16<T, false>(a[0]);
            fwd_get<T, M>(a[1], scr, j);
            fwd_put_s<T, M, 32>(a[2], tws, scr, j);
            dft16<T, false>(a[1]);
            fwd_get<T, M>(a[2], scr, j);
            dft16<T, false>(a[2]);
            // H^ = -N^ M^ ; rows of the folded tensor: sign -1 per folded odd axis
            mbar_wait(fullT, ph);
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                const int rs = rev16(s);
                const int kz = 2 * slot_freq<M>(j, s) + h;
                const bool up = rs > 8 || (rs == 8 && (j | h) != 0);
                const int kzf = up ? P - kz : kz;
                const T sz = up ? (T)-1 : (T)1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
                const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
                const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
                a[0][s] = mk<T>(-hx.x, -hx.y);
                a[1][s] = mk<T>(-hy.x, -hy.y);
                a[2][s] = mk<T>(-hz.x, -hz.y);
            }
            __syncwarp();
            if (lane == 0 && (arrive_count(cnt + 1) & 7) == 7) {  // every product is done: bring the next tile
                int ng = g, nsub = sub + 1;
                if (nsub >= nt) { ng = g + G; nsub = 0; }
                if (ng < nItems) {
                    mbar_expect_tx(fullB, S::TILE_BYTES);
                    bulk_load(s_B, tile_ptr(ng, nsub), S::TILE_BYTES, fullB);
                }
            }
            dft16<T, true>(a[0]);
            inv_put<T, M>(a[0], scr, j);
            dft16<T, true>(a[1]);
            inv_get_s<T, M, 32>(a[0], tws, scr, j);
            dft16<T, true>(a[2]);
            inv_put<T, M>(a[1], scr, j);
            dft16<T, true>(a[0]);
            inv_get_s<T, M, 32>(a[1], tws, scr, j);
            inv_put<T, M>(a[2], scr, j);
            dft16<T, true>(a[1]);
            inv_get_s<T, M, 32>(a[2], tws, scr, j);
            dft16<T, true>(a[2]);
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
            V *out = tile_ptr(g, sub) + coff;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {      // (fp64: half_sum's selects cost more registers than the kernel has)
                    V v = a[c][t];
                    v = cadd(v, shfl1(v));
                    if ((t >> 3) == h) out[(c * N + M * t) * TW] = v;
                }
            }
        }
    }
}

// ---- z pass, fp64, 128 cells along z -----------------------------------------------------------------
// k_pz_mid64 for M = 8: a team transforms two lines, so a warp owns two columns and four warps a tile;
// warps 0-3 take the +ky tile of an item and warps 4-7 the -ky tile (same folded tensor rows).  The
// region holds the tile pair (2 x 48 KB), then the tensor rows of the eight columns (48.75 KB).
struct Pz64Smem8 {
    static constexpr int N = 128;
    static constexpr int TILE_ELEMS = 3 * N * TW;                   // complex doubles
    static constexpr int TILE_BYTES = TILE_ELEMS * 16;              // 49152
    static constexpr int KZP = 130;
    static constexpr int TSLICE = 6 * KZP;
    static constexpr int TENS_BYTES = TW * TSLICE * 8;              // 49920, one bulk copy
    static constexpr int REGION = 2 * TILE_BYTES;
    static constexpr int OFF_SCR = REGION;
    static constexpr int SCR_BYTES = 16 * Team<8>::SCRATCH64 * 16;
    static constexpr int OFF_TW = OFF_SCR + SCR_BYTES;
    static constexpr int TW_BYTES = 16 * 32 * 16;
    static constexpr int OFF_BAR = OFF_TW + TW_BYTES;
    static constexpr int BYTES = OFF_BAR + 32;
};
static_assert(Pz64Smem8::BYTES <= 227 * 1024 && Pz64Smem8::TENS_BYTES <= Pz64Smem8::REGION, "k_pz_mid64_8 shared memory");

template <bool EMB>
__global__ void __launch_bounds__(kPipeThreads, 1)
k_pz_mid64_8(double2 *__restrict__ B, const double *__restrict__ Tn, int N2, int nItems, int kt0,
             const double2 *__restrict__ wP, int n3v)
{
    typedef double T;
    typedef double2 V;
    typedef Pz64Smem8 S;
    constexpr int M = 8, N = 128, P = 256;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_B = reinterpret_cast<V *>(smem);
    const T *s_T = reinterpret_cast<const T *>(smem);
    V *s_scr = reinterpret_cast<V *>(smem + S::OFF_SCR);
    V *s_tw = reinterpret_cast<V *>(smem + S::OFF_TW);
    uint64_t *fullB = reinterpret_cast<uint64_t *>(smem + S::OFF_BAR);
    uint64_t *fullT = fullB + 1;
    unsigned *cnt = reinterpret_cast<unsigned *>(fullT + 1);

    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int sub = w >> 2, cp = w & 3;
    const int h = lane & 1, i = lane >> 1;
    const int l = i >> 3, j = i & 7;
    const int k1 = 2 * cp + l;
    const int P2 = 2 * N2, K2 = N2 + 1;
    const int G = gridDim.x;

    auto tile_ptr = [&](int g, int sb) -> V * {
        const int kyf = g % K2, ktl = g / K2;
        const int ky = sb ? P2 - kyf : kyf;
        return B + ((long long)ktl * P2 + ky) * S::TILE_ELEMS;
    };
    auto n_tiles = [&](int g) -> int {
        const int kyf = g % K2;
        return (kyf == 0 || kyf == N2) ? 1 : 2;
    };
    auto load_item = [&](int g) {
        const int nt = n_tiles(g);
        mbar_expect_tx(fullB, nt * S::TILE_BYTES);
        for (int sb = 0; sb < nt; ++sb) bulk_load(s_B + sb * S::TILE_ELEMS, tile_ptr(g, sb), S::TILE_BYTES, fullB);
    };
    if (tid == 0) {
        mbar_init(fullB, 1);
        mbar_init(fullT, 1);
        cnt[0] = cnt[1] = 0;
        mbar_fence_init();
    }
    for (int q = tid; q < 16 * 32; q += kPipeThreads) {
        const int tp = q >> 5, ln = q & 31;
        s_tw[q] = wP[(((ln >> 1) & 7) * (2 * tp + (ln & 1))) & (P - 1)];
    }
    __syncthreads();
    if (tid == 0 && (int)blockIdx.x < nItems) load_item(blockIdx.x);
    const V *tws = s_tw + lane;
    V *scr = s_scr + (2 * w + h) * Team<M>::SCRATCH64;
    const T *ts = s_T + k1 * S::TSLICE;
    uint32_t ph = 0;

    for (int g = blockIdx.x; g < nItems; g += G, ph ^= 1) {
        const int kyf = g % K2, kt = kt0 + g / K2;
        const int nt = (kyf == 0 || kyf == N2) ? 1 : 2;
        const bool work = sub < nt;
        // element (c, e = j + 8 t) of column k1: row (c N + e), slot k1 ^ swz(e) ^ swz(ky); the fp64 swizzle of
        // e = j + 8 t is that of j for even t and 4 slots further for odd t
        const int cw = k1 ^ swzT<T>(sub ? P2 - kyf : kyf) ^ swzT<T>(j);
        const int offE = j * TW + cw, offO = j * TW + (cw ^ 4);
        mbar_wait(fullB, ph);
        V a[3][16];
        if (work) {
            const V *tb = s_B + sub * S::TILE_ELEMS;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    a[c][t] = tb[((t & 1) ? offO : offE) + (c * N + M * t) * TW];
                    if (EMB && j + M * t >= n3v) a[c][t] = mk<T>((T)0, (T)0);
                }
            }
        }
        __syncwarp();
        if (lane == 0 && (arrive_count(cnt) & 7) == 7) {
            mbar_expect_tx(fullT, S::TENS_BYTES);
            bulk_load(smem, Tn + ((long long)kt * K2 + kyf) * TW * S::TSLICE, S::TENS_BYTES, fullT);
        }
        if (work) {
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, false>(a[c]);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                dft16<T, false>(a[c]);
                fwd_put_s<T, M, 32>(a[c], tws, scr, i);
                fwd_get<T, M>(a[c], scr, i);
                dftM<T, false, M>(a[c]);
            }
        }
        mbar_wait(fullT, ph);
        if (work) {
            const T sy = sub ? (T)-1 : (T)1;
#pragma unroll
            for (int s = 0; s < 16; ++s) {
                const int u = s / M, r8 = rev8(s % M);
                const int kz = 2 * slot_freq<M>(j, s) + h;
                const bool up = r8 > 4 || (r8 == 4 && (j | u | h) != 0);
                const int kzf = up ? P - kz : kz;
                const T sz = up ? (T)-1 : (T)1;
                const T *tp = ts + kzf;
                const T nxx = tp[0], nyy = tp[S::KZP], nzz = tp[2 * S::KZP];
                const T nxy = sy * tp[3 * S::KZP], nxz = sz * tp[4 * S::KZP], nyz = sy * sz * tp[5 * S::KZP];
                const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
                const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
                const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
                const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
                a[0][s] = mk<T>(-hx.x, -hx.y);
                a[1][s] = mk<T>(-hy.x, -hy.y);
                a[2][s] = mk<T>(-hz.x, -hz.y);
            }
        }
        __syncwarp();
        if (lane == 0 && (arrive_count(cnt + 1) & 7) == 7 && g + G < nItems) load_item(g + G);
        if (work) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                dftM<T, true, M>(a[c]);
                inv_put<T, M>(a[c], scr, i);
                inv_get_s<T, M, 32>(a[c], tws, scr, i);
                dft16<T, true>(a[c]);
            }
            if (h) {
#pragma unroll
                for (int c = 0; c < 3; ++c) shift32<T, true>(a[c]);
            }
            V *out = tile_ptr(g, sub);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    V v = a[c][t];
                    v = cadd(v, shfl1(v));
                    if ((t >> 3) == h) out[((t & 1) ? offO : offE) + (c * N + M * t) * TW] = v;
                }
            }
        }
    }
}


// ---- x passes ----------------------------------------------------------------------------------
// Geometry shared by k_px_fwd / k_px_inv for N1 = 16 M: a CTA of 8 warps owns R = 2 LINES cell rows
// (c2) of one cell plane c3; warp w transforms LINES/8 = 16/M complex lines, each packing the two
// real rows 2 line, 2 line + 1.  The half spectrum has NKT = 2 M + 1 tiles of 8 columns.
template <typename T, int M> struct PxGeom {
    static constexpr int N = 16 * M, P = 2 * N, LT = 16 / M;
    static constexpr int LINES = 8 * LT, R = 2 * LINES;
    static constexpr int NKT = 2 * M + 1;
    static constexpr int YP = N + 2;            // pitch of the y-summed node rows (row pairs)
    static constexpr int PZ = P + 8;            // pitch of a packed spectrum line
    static constexpr int SCR = team_scratch<T, M>();
    static constexpr size_t FWD_BYTES = ((size_t)LINES * YP + (size_t)LINES * PZ + 16 * SCR) * 2 * sizeof(T);
    // forward, bulk-fed (M >= 4): the packed lines of a warp live in that warp's own exchange scratch
    // (LT PZ <= 2 SCR), and a raw buffer takes the R + 1 node rows of the two planes of the next component
    static constexpr bool BULK_OK = LT * PZ <= 2 * SCR;     // M >= 4
    static constexpr int AL = 16 / (int)sizeof(T);          // elements per 16 bytes: bulk copies start and end on these
    __host__ __device__ static constexpr int raw_pitch(int n1) { return ((R + 1) * n1 + 6 + 31) & ~31; }     // reals per plane
    static size_t fwd_bulk_bytes(int n1) { return ((size_t)LINES * YP + 16 * SCR) * 2 * sizeof(T) + (size_t)2 * raw_pitch(n1) * sizeof(T) + 16; }
    // inverse: output tile (R x N reals) + exchange scratch + staged spectrum rows of one component, the
    // blocks of consecutive k1 tiles 64 bytes apart modulo 128 (the gather of a half-warp spans two)
    static constexpr int SK = 64 / (2 * (int)sizeof(T));    // 64 bytes of complex elements
    static constexpr int KP = R * 8 + SK;                   // pitch of a staged k1 tile
    static constexpr size_t INV_BYTES = (size_t)R * N * sizeof(T) + ((size_t)16 * SCR + (size_t)NKT * KP) * 2 * sizeof(T);
};

template <typename V> __device__ __forceinline__ void store2(V *dst, V a, V b);
template <> __device__ __forceinline__ void store2<float2>(float2 *dst, float2 a, float2 b)
{
    *reinterpret_cast<float4 *>(dst) = make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ void store2<double2>(double2 *dst, double2 a, double2 b)
{
    // one 32-byte store (sm_100: 256-bit global vector access; dst is 32-byte aligned): two 16-byte stores would each
    // fill half a sector, and the store queue is what this loop waits on in fp64
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(dst), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y) : "memory");
}
template <typename V> __device__ __forceinline__ void load2(const V *src, V &a, V &b);
template <> __device__ __forceinline__ void load2<float2>(const float2 *src, float2 &a, float2 &b)
{
    const float4 v = *reinterpret_cast<const float4 *>(src);
    a = make_float2(v.x, v.y);
    b = make_float2(v.z, v.w);
}
template <> __device__ __forceinline__ void load2<double2>(const double2 *src, double2 &a, double2 &b)
{
    a = src[0];
    b = src[1];
}

// x forward (a1 + the x part of a2): M_c = Ms_c (1/8) sum of the 8 vertices, two real cell rows per
// complex line, padded transform, untangle, blocked swizzled store A[kt][comp][c3][c2][8].
//   phase 1  thread = node column, marches over 17 node rows adding the two planes (z) and
//            consecutive rows (y): ys2[line][n1] = (row 2 line, row 2 line + 1)
//   phase 2  cell value = Ms/8 (ys2[e] + ys2[e+1]) on the way into the registers; transform
//   phase 3  Xa[k] = (Z[k] + conj Z[P-k])/2, Xb[k] = (Z[k] - conj Z[P-k])/(2i), both rows of a line
//            by one thread, 16-byte stores
// EMB (embedded mesh, nm_fast_plan): the mesh has N1 <= N cells per row; cells beyond it are zero, node
// columns beyond n1 are not read, and the rows of A have pitch f2 (the y transform extent) >= N2.
// BULK (M >= 4, 16-byte aligned field): the node rows of a component -- R + 1 contiguous rows in each of the
// two planes -- arrive by two bulk copies issued one component ahead (from the 16-byte boundary below their
// start: `shift` elements into the buffer), so phase 1 reads shared memory and the HBM latency is off the path.
template <typename T, int M, bool UNI, bool EMB, bool BULK>
__global__ void __launch_bounds__(kPipeThreads, sizeof(T) == 8 ? 1 : 2)
k_px_fwd(const T *__restrict__ fld, const T *__restrict__ Ms, T ms_uni, typename VT<T>::V *__restrict__ A,
         NmGeom g, const typename VT<T>::V *__restrict__ wP, int f2, int persist)
{
    typedef typename VT<T>::V V;
    typedef PxGeom<T, M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, LINES = G::LINES, R = G::R, NKT = G::NKT;
    static_assert(!BULK || G::BULK_OK, "bulk-fed x pass: M >= 4");
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_y = reinterpret_cast<V *>(smem);                   // LINES x YP
    V *s_z = s_y + LINES * G::YP;                           // LINES x PZ (BULK: inside the scratch, per warp)
    V *s_scr = BULK ? s_z : s_z + LINES * G::PZ;
    const int RP = G::raw_pitch(g.n1);
    T *s_raw = reinterpret_cast<T *>(s_scr + 16 * G::SCR);  // BULK: 2 planes x RP
    uint64_t *full = reinterpret_cast<uint64_t *>(s_raw + 2 * RP);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = i / M, j = i % M;
    const int line = w * LT + l;
    // persist (BULK only): a CTA walks the tiles blockIdx.x, blockIdx.x + gridDim.x, ... (tile = row block + nbx * plane)
    // and requests the first component of its next tile while the last one of this tile is transformed
    int r0 = blockIdx.x * R, c3 = blockIdx.y;
    const int nbx = g.N2 / R, ntiles = persist ? nbx * g.N3 : 1;
    V *scr = s_scr + (2 * w + h) * G::SCR;
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    // Ms/8 of this thread's cells (rows 2 line, 2 line + 1; columns e = j + M t)
    constexpr bool MS1 = UNI && !EMB;                       // one Ms/8 for every cell of the thread
    V msr[MS1 ? 1 : 16];
    auto load_ms = [&]() {
        if (MS1) { msr[0] = mk<T>((T)0.125 * ms_uni, (T)0.125 * ms_uni); return; }
        const int N1 = EMB ? g.N1 : N;
        const T *mrow = Ms + ((long long)c3 * g.N2 + r0 + 2 * line) * N1 + j;
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            V v;
            if (EMB && j + M * t >= N1) v = mk<T>((T)0, (T)0);
            else if (UNI) v = mk<T>((T)0.125 * ms_uni, (T)0.125 * ms_uni);
            else v = mk<T>((T)0.125 * mrow[M * t], (T)0.125 * mrow[N1 + M * t]);
            msr[MS1 ? 0 : t] = v;
        }
    };
    const long long plane = (long long)g.n1 * g.n2;
    const int rg = tid / N, col = tid % N;                  // phase 1: row group (16 cell rows) and node column
    // small grids: the three components in three CTAs (gridDim.z = 3)
    const int comp_lo = gridDim.z == 3 ? blockIdx.z : 0, comp_hi = gridDim.z == 3 ? comp_lo + 1 : 3;
    // z sums of component `comp`: 17 node rows of this thread's column, and (threads < R) the last node column;
    // in fp64 (one CTA per SM) those of component comp + 1 are requested before component comp is
    // transformed, so that they travel while the SM computes
    T z[17], zlast = (T)0;
    auto load_z = [&](int comp) {
        const T *base = fld + (long long)comp * g.nodes + (long long)c3 * plane + (long long)(r0 + rg * 16) * g.n1;
#pragma unroll
        for (int r = 0; r < 17; ++r)
            z[r] = (!EMB || col < g.n1) ? base[(long long)r * g.n1 + col] + base[plane + (long long)r * g.n1 + col] : (T)0;
        if (tid < R) {   // last node column n1 = N
            const T *q = fld + (long long)comp * g.nodes + (long long)c3 * plane + (long long)(r0 + tid) * g.n1 + N;
            zlast = (!EMB || N < g.n1) ? (q[0] + q[plane]) + (q[g.n1] + q[plane + g.n1]) : (T)0;
        }
    };
    constexpr bool PREF = sizeof(T) == 8 && !BULK;          // register prefetch: the fp64 form without the raw-row buffer (fp32: measured slower)
    // BULK: thread 0 requests the rows of a component; element e0 of the array lands at s_raw[p RP + (e0 & (AL - 1))]
    const int nodes3 = 3 * (int)g.nodes;
    auto request = [&](int comp, int rr0, int cc3) {
        int e0[2], len[2], total = 0;
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const int e = comp * (int)g.nodes + (cc3 + p) * (int)plane + rr0 * g.n1;
            e0[p] = e & ~(G::AL - 1);
            len[p] = ((R + 1) * g.n1 + (e & (G::AL - 1)) + G::AL - 1) & ~(G::AL - 1);
            if (e0[p] + len[p] > nodes3) {                  // the array ends inside the last 16 bytes: its last elements by hand
                len[p] = (nodes3 - e0[p]) & ~(G::AL - 1);
                for (int q = e0[p] + len[p]; q < nodes3; ++q) s_raw[p * RP + q - e0[p]] = fld[q];
            }
            total += len[p];
        }
        mbar_expect_tx(full, (uint32_t)(total * sizeof(T)));
#pragma unroll
        for (int p = 0; p < 2; ++p) bulk_load(s_raw + p * RP, fld + e0[p], (uint32_t)(len[p] * sizeof(T)), full);
    };
    auto take_z = [&](int comp) {
        const int sh0 = (comp * (int)g.nodes + c3 * (int)plane + r0 * g.n1) & (G::AL - 1);
        const int sh1 = (comp * (int)g.nodes + (c3 + 1) * (int)plane + r0 * g.n1) & (G::AL - 1);
        const T *q0 = s_raw + sh0 + rg * 16 * g.n1 + col, *q1 = s_raw + RP + sh1 + rg * 16 * g.n1 + col;
#pragma unroll
        for (int r = 0; r < 17; ++r) z[r] = (!EMB || col < g.n1) ? q0[r * g.n1] + q1[r * g.n1] : (T)0;
        if (tid < R) {
            const T *a0 = s_raw + sh0 + tid * g.n1 + N, *a1 = s_raw + RP + sh1 + tid * g.n1 + N;
            zlast = (!EMB || N < g.n1) ? (a0[0] + a1[0]) + (a0[g.n1] + a1[g.n1]) : (T)0;
        }
    };
    unsigned nwait = 0;
    if (BULK) {
        if (tid == 0) {
            mbar_init(full, 1);
            mbar_fence_init();
        }
        __syncthreads();
        if (persist) { r0 = ((int)blockIdx.x % nbx) * R; c3 = (int)blockIdx.x / nbx; }
        if (tid == 0) request(comp_lo, r0, c3);
    }
    for (int tile = persist ? (int)blockIdx.x : 0; tile < ntiles; tile += persist ? (int)gridDim.x : 1) {
    if (persist) { r0 = (tile % nbx) * R; c3 = tile / nbx; }
    load_ms();
    if (PREF) load_z(comp_lo);
    for (int comp = comp_lo; comp < comp_hi; ++comp) {
        if (BULK) {
            mbar_wait(full, nwait & 1u);
            ++nwait;
            take_z(comp);
        } else if (!PREF) load_z(comp);
#pragma unroll
        for (int r = 0; r < 16; r += 2)
            s_y[(rg * 8 + (r >> 1)) * G::YP + col] = mk<T>(z[r] + z[r + 1], z[r + 1] + z[r + 2]);
        if (tid < R) reinterpret_cast<T *>(s_y + (tid >> 1) * G::YP + N)[tid & 1] = zlast;
        __syncthreads();
        if (BULK && tid == 0) {                             // the raw rows have been read by everyone
            const int nt = tile + (int)gridDim.x;
            if (comp + 1 < comp_hi) request(comp + 1, r0, c3);
            else if (persist && nt < ntiles) request(comp_lo, (nt % nbx) * R, nt / nbx);
        }
        if (PREF && comp + 1 < comp_hi) load_z(comp + 1);
        V a[16];
        const V *yl = s_y + line * G::YP + j;
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const V v0 = yl[M * t], v1 = yl[M * t + 1];
            const V mm = msr[MS1 ? 0 : t];
            a[t] = mk<T>(mm.x * (v0.x + v1.x), mm.y * (v0.y + v1.y));
        }
        if (h) shift32<T, false>(a);
        fft_fwd<T, M, true>(a, tw, scr, i);
        // packed line `ln`: BULK keeps the LT lines of warp ln / LT in that warp's two exchange scratches
        auto zline = [&](int ln) -> V * { return BULK ? s_scr + (ln / LT) * 2 * G::SCR + (ln % LT) * G::PZ : s_z + ln * G::PZ; };
        if (BULK) __syncwarp();                             // every lane has taken its values out of the scratch
        {
            V *zw = zline(line);
#pragma unroll
            for (int s = 0; s < 16; ++s) zw[2 * slot_freq<M>(j, s) + h] = a[s];
        }
        __syncthreads();
        for (int idx = tid; idx < NKT * LINES * 4; idx += kPipeThreads) {
            const int q = idx & 3, ln = (idx >> 2) % LINES, kt = idx / (4 * LINES);
            const int c2 = r0 + 2 * ln;
            const int p0 = 2 * q;                           // physical slots p0, p0 + 1 of the blocked row
            const int k0 = kt * TW + (p0 ^ swzT<T>(c2)), k1 = k0 ^ 1;
            const V *zl = zline(ln);
            V ze, zo;
            load2(zl + (k0 & ~1), ze, zo);
            const V za = (k0 & 1) ? zo : ze, zb = (k0 & 1) ? ze : zo;      // Z[k0], Z[k1]
            const V ma = zl[(P - k0) & (P - 1)], mb = zl[(P - k1) & (P - 1)];
            const T hf = (T)0.5;
            V a0 = mk<T>(hf * (za.x + ma.x), hf * (za.y - ma.y)), b0 = mk<T>(hf * (za.y + ma.y), hf * (ma.x - za.x));
            V a1 = mk<T>(hf * (zb.x + mb.x), hf * (zb.y - mb.y)), b1 = mk<T>(hf * (zb.y + mb.y), hf * (mb.x - zb.x));
            if (k0 > N) { a0 = mk<T>((T)0, (T)0); b0 = a0; }
            if (k1 > N) { a1 = mk<T>((T)0, (T)0); b1 = a1; }
            V *dst = A + ((((long long)kt * 3 + comp) * g.N3 + c3) * f2 + c2) * TW + p0;
            store2(dst, a0, a1);
            // row c2 + 1 (c2 even): the same columns; its fp64 swizzle differs in slot bit 2
            store2(dst + TW + (sizeof(T) == 8 ? (p0 ^ 4) - p0 : 0), b0, b1);
        }
    }
    }
}

// x inverse (the x part of a4): rebuild the packed spectrum Z = Xa + i Xb of two real rows from their
// half spectra (Z[P-k] = conj Xa[k] + i conj Xb[k]), inverse transform cropped to N1, write the cell
// field Hc[comp][c3][c2][c1] through a row-major staging tile with 16-byte stores.
// The spectrum rows of a component are NKT contiguous blocks of R rows x 8 columns; cp.async brings
// the blocks of component c + 1 into a raw staging buffer while component c is transformed and
// stored, so the global-load latency of a CTA is hidden behind its own arithmetic (the output tile
// aliases the packed-line buffer, which keeps two CTAs per SM in fp32).
template <typename T, int M, bool EMB>
__global__ void __launch_bounds__(kPipeThreads, sizeof(T) == 8 ? 1 : 2)
k_px_inv(const typename VT<T>::V *__restrict__ A, T *__restrict__ Hc, NmGeom g, const typename VT<T>::V *__restrict__ wP,
         int f2, int persist)
{
    typedef typename VT<T>::V V;
    typedef PxGeom<T, M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, R = G::R, NKT = G::NKT;
    extern __shared__ __align__(1024) unsigned char smem[];
    T *s_out = reinterpret_cast<T *>(smem);                 // output tile R x N (reals)
    V *s_scr = reinterpret_cast<V *>(smem + (size_t)R * N * sizeof(T));
    V *s_raw = s_scr + 16 * G::SCR;                         // NKT blocks of R x 8 staged spectrum rows (pitch KP)
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = i / M, j = i % M;
    const int line = w * LT + l;
    // persist: a CTA walks the tiles blockIdx.x, blockIdx.x + gridDim.x, ... (tile = row block + nbx * plane) and
    // stages the first component of its next tile while the last one of this tile is transformed
    int r0 = blockIdx.x * R, c3 = blockIdx.y;
    const int nbx = g.N2 / R, ntiles = persist ? nbx * g.N3 : 1;
    if (persist) { r0 = ((int)blockIdx.x % nbx) * R; c3 = (int)blockIdx.x / nbx; }
    V *scr = s_scr + (2 * w + h) * G::SCR;
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    constexpr int PIECES = R * TW * (int)sizeof(V) / 16;    // 16-byte pieces per block
    auto stage = [&](int comp, int rr0, int cc3) {
        for (int e = tid; e < NKT * PIECES; e += kPipeThreads) {
            const int kt = e / PIECES, off = e - kt * PIECES;
            const char *src = reinterpret_cast<const char *>(A + ((((long long)kt * 3 + comp) * g.N3 + cc3) * f2 + rr0) * TW) + off * 16;
            const unsigned dst = smem_u32(reinterpret_cast<char *>(s_raw + kt * G::KP) + off * 16);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int comp_lo = gridDim.z == 3 ? blockIdx.z : 0, comp_hi = gridDim.z == 3 ? comp_lo + 1 : 3;
    stage(comp_lo, r0, c3);
    // Xa, Xb of this thread's line: rows 2 line, 2 line + 1 of every block, column k1 at slot k1 ^ swz(c2)
    const V *ra = s_raw + (2 * line) * TW;
    for (int tile = persist ? (int)blockIdx.x : 0; tile < ntiles; tile += persist ? (int)gridDim.x : 1) {
    if (persist) { r0 = (tile % nbx) * R; c3 = tile / nbx; }
    const int sw = swzT<T>(r0 + 2 * line);
    for (int comp = comp_lo; comp < comp_hi; ++comp) {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                                    // staged rows visible; the output tile has been read
        // packed spectrum of the two rows, gathered straight into transform order:
        //   Z[k] = Xa[k] + i Xb[k] (k <= N),   Z[k] = conj Xa[P-k] + i conj Xb[P-k] (k > N)
        V a[16];
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int k = 2 * slot_freq<M>(j, s) + h;
            const bool up = k > N;
            const int kk = up ? P - k : k;
            const V *q = ra + (kk >> 3) * G::KP + ((kk & 7) ^ sw);
            const V u = q[0], v = (sizeof(T) == 8 ? ra + (kk >> 3) * G::KP + ((kk & 7) ^ sw ^ 4) : q)[TW];   // row + 1: fp64 slot bit 2
            const T sg = up ? (T)-1 : (T)1;
            a[s] = mk<T>(u.x - sg * v.y, v.x + sg * u.y);
        }
        __syncthreads();                                    // the staging buffer is free
        if (comp + 1 < comp_hi) stage(comp + 1, r0, c3);
        else if (persist && tile + (int)gridDim.x < ntiles) stage(comp_lo, ((tile + (int)gridDim.x) % nbx) * R, (tile + (int)gridDim.x) / nbx);
        fft_inv<T, M, true>(a, tw, scr, i);
        if (h) shift32<T, true>(a);
        if (M >= 8) {
            // straight to Hc: in one store the 16 (M = 16) or 8 lanes of a line cover 64 / 32 contiguous
            // bytes of a cell row; half h of a thread stores elements j + M (tt + 8 h)
            const int n1row = EMB ? g.N1 : N;
            T *rowA = Hc + (long long)comp * g.cells + ((long long)c3 * g.N2 + r0 + 2 * line) * n1row;
#pragma unroll
            for (int tt = 0; tt < 8; ++tt) {
                const V v = half_sum(a, tt, h);
                const int e = j + M * (tt + 8 * h);
                if (!EMB || e < n1row) {
                    rowA[e] = v.x;
                    rowA[n1row + e] = v.y;
                }
            }
        } else {
            // short lines: through a row-major staging tile, 16-byte stores
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                const V v = half_sum(a, s, h);
                s_out[(2 * line) * N + j + M * (s + 8 * h)] = v.x;
                s_out[(2 * line + 1) * N + j + M * (s + 8 * h)] = v.y;
            }
            __syncthreads();
            constexpr int VEC = 16 / sizeof(T);
            if (!EMB) {     // R consecutive rows of Hc are contiguous
                T *dst = Hc + (long long)comp * g.cells + ((long long)c3 * g.N2 + r0) * N;
                for (int idx = tid; idx < R * N / VEC; idx += kPipeThreads)
                    reinterpret_cast<int4 *>(dst)[idx] = reinterpret_cast<const int4 *>(s_out)[idx];
            } else {        // rows of N1 <= N cells (N1 a multiple of 4): the first N1 columns of every tile row
                const int pr = g.N1 / VEC;
                T *dst = Hc + (long long)comp * g.cells + ((long long)c3 * g.N2 + r0) * g.N1;
                for (int idx = tid; idx < R * pr; idx += kPipeThreads) {
                    const int row = idx / pr, cv = idx - row * pr;
                    reinterpret_cast<int4 *>(dst)[idx] = reinterpret_cast<const int4 *>(s_out)[row * (N / VEC) + cv];
                }
            }
        }
    }
    }
}


// ---- y passes ----------------------------------------------------------------------------------
// Tile = one (k1 tile, component, c3): the A side is a contiguous [c2 = 256][8] block (one bulk
// copy), the B side is 512 rows of 64 bytes, one per ky, 3 N3 rows apart: a 4-D tensor map over
// B[kt P2 + ky][comp][c3][16 floats] moves them as two boxes of 256 rows.  Persistent CTAs, two per
// SM; thread 0 keeps the copies of the neighbouring tiles in flight around the transform.
template <typename T> struct PySmem {
    typedef typename VT<T>::V V;
    static constexpr int N = 256, P = 512;
    static constexpr int A_ELEMS = N * TW, A_BYTES = A_ELEMS * (int)sizeof(V);         // 16384 (fp32) / 32768
    static constexpr int B_ELEMS = P * TW, B_BYTES = B_ELEMS * (int)sizeof(V);         // 32768 / 65536
    static constexpr int SCR_BYTES = 16 * team_scratch<T, 16>() * (int)sizeof(V);      // 35840 / 70656
    // forward: two A stages in, one B tile out; inverse: one B stage in (reloaded as soon as it is read), one A tile out
    static constexpr int FWD_BYTES = 2 * A_BYTES + B_BYTES + SCR_BYTES + 64;
    static constexpr int INV_BYTES = B_BYTES + A_BYTES + SCR_BYTES + 64;
    static constexpr int CTAS = sizeof(T) == 8 ? 1 : 2;                                // persistent CTAs per SM
};
static_assert(PySmem<double>::FWD_BYTES <= 227 * 1024, "k_py_fwd<double> shared memory exceeds the sm_100a per-CTA limit");

// EMB: rows c2 >= n2v of an A tile were never written (embedded mesh) and enter as zeros.
template <typename T, bool EMB>
__global__ void __launch_bounds__(kPipeThreads, PySmem<T>::CTAS)
k_py_fwd(const typename VT<T>::V *__restrict__ A, const __grid_constant__ NmTensorMap tmB, int N3, int nTiles, int kt0,
         const typename VT<T>::V *__restrict__ wP, int n2v)
{
    typedef typename VT<T>::V V;
    typedef PySmem<T> S;
    constexpr int M = 16;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_out = reinterpret_cast<V *>(smem);                                 // [P][8]
    V *s_in = reinterpret_cast<V *>(smem + S::B_BYTES);                     // 2 x [N][8]
    V *s_scr = reinterpret_cast<V *>(smem + S::B_BYTES + 2 * S::A_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S::B_BYTES + 2 * S::A_BYTES + S::SCR_BYTES);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, j = lane >> 1;
    const int G = gridDim.x;
    if (tid == 0) {
        mbar_init(full, 1);
        mbar_init(full + 1, 1);
        mbar_fence_init();
        tensormap_prefetch(&tmB);
    }
    __syncthreads();
    // tile tl -> (ktl, comp, c3), c3 fastest: consecutive tiles are consecutive 16 KB blocks of A
    auto a_tile = [&](int tl) -> const V * { return A + ((long long)kt0 * 3 * N3 + tl) * S::A_ELEMS; };
    if (tid == 0) {
        for (int q = 0; q < 2; ++q) {
            const int tl = blockIdx.x + q * G;
            if (tl < nTiles) {
                mbar_expect_tx(full + q, S::A_BYTES);
                bulk_load(s_in + q * S::A_ELEMS, a_tile(tl), S::A_BYTES, full + q);
            }
        }
    }
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + (2 * w + h) * team_scratch<T, M>();
    const int cin = j * TW + (w ^ swzT<T>(j));              // A rows are swizzled by c2 = e, swz(j + 16 t) = swz(j)
    int n = 0;
    for (int tl = blockIdx.x; tl < nTiles; tl += G, ++n) {
        const int c3 = tl % N3, comp = (tl / N3) % 3, ktl = tl / (3 * N3);
        const int b = n & 1;
        mbar_wait(full + b, (uint32_t)((n >> 1) & 1));
        const V *in = s_in + b * S::A_ELEMS + cin;
        V a[16];
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            a[t] = in[M * t * TW];
            if (EMB && j + M * t >= n2v) a[t] = mk<T>((T)0, (T)0);
        }
        __syncthreads();                                    // stage b is free again
        if (tid == 0 && tl + 2 * G < nTiles) {
            mbar_expect_tx(full + b, S::A_BYTES);
            bulk_load(s_in + b * S::A_ELEMS, a_tile(tl + 2 * G), S::A_BYTES, full + b);
        }
        if (h) shift32<T, false>(a);
        fft_fwd<T, M, true>(a, tw, scr, j);
        if (tid == 0) bulk_wait_read<0>();                  // the previous tile has left s_out
        __syncthreads();
        // row ky = 2 (j + 16 rev16(s)) + h, column k1 = w swizzled by c3 and ky: swz(ky) = swz(2 j + h)
        V *out = s_out + (2 * j + h) * TW + (w ^ swzT<T>(c3) ^ swzT<T>(2 * j + h));
#pragma unroll
        for (int s = 0; s < 16; ++s) out[32 * rev16(s) * TW] = a[s];
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            tensor_store_4d(&tmB, s_out, 0, c3, comp, ktl * S::P);
            tensor_store_4d(&tmB, s_out + 256 * TW, 0, c3, comp, ktl * S::P + 256);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait<0>();
}

template <typename T>
__global__ void __launch_bounds__(kPipeThreads, PySmem<T>::CTAS)
k_py_inv(const __grid_constant__ NmTensorMap tmB, typename VT<T>::V *__restrict__ A, int N3, int nTiles, int kt0,
         const typename VT<T>::V *__restrict__ wP)
{
    typedef typename VT<T>::V V;
    typedef PySmem<T> S;
    constexpr int M = 16;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_in = reinterpret_cast<V *>(smem);                                  // [P][8]
    V *s_out = reinterpret_cast<V *>(smem + S::B_BYTES);                    // [N][8]
    V *s_scr = reinterpret_cast<V *>(smem + S::B_BYTES + S::A_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S::B_BYTES + S::A_BYTES + S::SCR_BYTES);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, j = lane >> 1;
    const int G = gridDim.x;
    if (tid == 0) {
        mbar_init(full, 1);
        mbar_fence_init();
        tensormap_prefetch(&tmB);
    }
    __syncthreads();
    auto load_b = [&](int tl) {
        const int c3 = tl % N3, comp = (tl / N3) % 3, ktl = tl / (3 * N3);
        mbar_expect_tx(full, S::B_BYTES);
        tensor_load_4d(s_in, &tmB, 0, c3, comp, ktl * S::P, full);
        tensor_load_4d(s_in + 256 * TW, &tmB, 0, c3, comp, ktl * S::P + 256, full);
    };
    if (tid == 0 && (int)blockIdx.x < nTiles) load_b(blockIdx.x);
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + (2 * w + h) * team_scratch<T, M>();
    const int cout = j * TW + (w ^ swzT<T>(j));
    int n = 0;
    for (int tl = blockIdx.x; tl < nTiles; tl += G, ++n) {
        const int c3 = tl % N3;
        mbar_wait(full, (uint32_t)(n & 1));
        const V *in = s_in + (2 * j + h) * TW + (w ^ swzT<T>(c3) ^ swzT<T>(2 * j + h));
        V a[16];
#pragma unroll
        for (int s = 0; s < 16; ++s) a[s] = in[32 * rev16(s) * TW];
        __syncthreads();                                    // the stage is free again
        if (tid == 0 && tl + G < nTiles) load_b(tl + G);
        fft_inv<T, M, true>(a, tw, scr, j);
        if (h) shift32<T, true>(a);
        if (tid == 0) bulk_wait_read<0>();                  // the previous tile has left s_out
        __syncthreads();
        V *out = s_out + cout;
#pragma unroll
        for (int s = 0; s < 8; ++s) out[M * (s + 8 * h) * TW] = half_sum(a, s, h);
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            bulk_store(A + ((long long)kt0 * 3 * N3 + tl) * S::A_ELEMS, s_out, S::A_BYTES);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait<0>();
}

// ---- y passes, 128 cells along y ---------------------------------------------------------------------
// M = 8: a team transforms two lines, here the planes c3_0, c3_0 + 1 of one (k1 tile, component); the
// warps are the eight columns as before.  A side: two contiguous [128][8] blocks (8 KB each), the
// second one staged 16 bytes further so that the two lines of a half-warp use different banks.
// B side: 256 rows of 128 bytes (ky; both planes), one 4-D box.  Lane = (j, line, half) with the line
// in bit 1, so that a half-warp scatters into both 64-byte halves of the B rows (the slot parity of
// an output is the same for every lane, which leaves a two-way conflict on that side).
template <typename T> struct Py8Smem {
    typedef typename VT<T>::V V;
    static constexpr int N = 128, P = 256;
    static constexpr int LINE_ELEMS = N * TW;                               // 1024 complex, 8 KB (fp32) / 16 KB
    static constexpr int A_ELEMS = 2 * LINE_ELEMS + 16;                     // two lines, 2 elements of skew, padded to 128 B
    static constexpr int A_BYTES = A_ELEMS * (int)sizeof(V);
    static constexpr int B_ELEMS = P * 2 * TW, B_BYTES = B_ELEMS * (int)sizeof(V);   // 32768 / 65536
    static constexpr int SCR_BYTES = 16 * team_scratch<T, 8>() * (int)sizeof(V);
    static constexpr int FWD_BYTES = 2 * A_BYTES + B_BYTES + SCR_BYTES + 64;
    static constexpr int INV_BYTES = B_BYTES + A_BYTES + SCR_BYTES + 64;
    static constexpr int CTAS = sizeof(T) == 8 ? 1 : 2;
};
static_assert(Py8Smem<double>::FWD_BYTES <= 227 * 1024, "k_py_fwd8<double> shared memory exceeds the sm_100a per-CTA limit");

template <typename T, bool EMB>
__global__ void __launch_bounds__(kPipeThreads, Py8Smem<T>::CTAS)
k_py_fwd8(const typename VT<T>::V *__restrict__ A, const __grid_constant__ NmTensorMap tmB, int N3, int nTiles, int kt0,
          const typename VT<T>::V *__restrict__ wP, int n2v)
{
    typedef typename VT<T>::V V;
    typedef Py8Smem<T> S;
    constexpr int M = 8;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_out = reinterpret_cast<V *>(smem);                                 // [P][2][8]
    V *s_in = reinterpret_cast<V *>(smem + S::B_BYTES);                     // 2 stages
    V *s_scr = reinterpret_cast<V *>(smem + S::B_BYTES + 2 * S::A_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S::B_BYTES + 2 * S::A_BYTES + S::SCR_BYTES);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, l = (lane >> 1) & 1, j = lane >> 2, i = l * M + j;
    const int G = gridDim.x, H3 = N3 / 2;
    if (tid == 0) {
        mbar_init(full, 1);
        mbar_init(full + 1, 1);
        mbar_fence_init();
        tensormap_prefetch(&tmB);
    }
    __syncthreads();
    // tile tl -> (ktl, comp, plane pair q), q fastest: consecutive tiles are consecutive 16 KB of A
    auto load_a = [&](int tl, int b) {
        const V *src = A + ((long long)kt0 * 3 * H3 + tl) * 2 * S::LINE_ELEMS;
        mbar_expect_tx(full + b, 2 * S::LINE_ELEMS * (int)sizeof(V));
        bulk_load(s_in + b * S::A_ELEMS, src, S::LINE_ELEMS * (int)sizeof(V), full + b);
        bulk_load(s_in + b * S::A_ELEMS + S::LINE_ELEMS + 2, src + S::LINE_ELEMS, S::LINE_ELEMS * (int)sizeof(V), full + b);
    };
    if (tid == 0) {
        for (int q = 0; q < 2; ++q)
            if ((int)blockIdx.x + q * G < nTiles) load_a(blockIdx.x + q * G, q);
    }
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + (2 * w + h) * team_scratch<T, M>();
    // element e = j + 8 t of line l: row e, slot w ^ swz(e), swz(j + 8 t) = swz(j) ^ 4 (t & 1)
    const int cinE = l * (S::LINE_ELEMS + 2) + j * TW + (w ^ swzT<T>(j));
    const int cinO = l * (S::LINE_ELEMS + 2) + j * TW + (w ^ swzT<T>(j) ^ 4);
    int n = 0;
    for (int tl = blockIdx.x; tl < nTiles; tl += G, ++n) {
        const int q = tl % H3, comp = (tl / H3) % 3, ktl = tl / (3 * H3);
        const int c3_0 = 2 * q;
        const int b = n & 1;
        mbar_wait(full + b, (uint32_t)((n >> 1) & 1));
        const V *in = s_in + b * S::A_ELEMS;
        V a[16];
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            a[t] = in[((t & 1) ? cinO : cinE) + M * t * TW];
            if (EMB && j + M * t >= n2v) a[t] = mk<T>((T)0, (T)0);
        }
        __syncthreads();                                    // stage b is free again
        if (tid == 0 && tl + 2 * G < nTiles) load_a(tl + 2 * G, b);
        if (h) shift32<T, false>(a);
        fft_fwd<T, M, true>(a, tw, scr, i);
        if (tid == 0) bulk_wait_read<0>();                  // the previous tile has left s_out
        __syncthreads();
        // slot s = 8 u + p holds ky = 2 (2 j + u + 16 rev8(p)) + h; element (ky, l): row 2 ky + l,
        // column w swizzled by the plane and by ky: swz(ky) = swz(4 j + 2 u + h)
        const int cs = w ^ swzT<T>(c3_0 + l);          // plane c3_0 + l of the pair
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int u = s / M, r8 = rev8(s % M);
            const int ky = 4 * j + 2 * u + 32 * r8 + h;
            s_out[(2 * ky + l) * TW + (cs ^ swzT<T>(4 * j + 2 * u + h))] = a[s];
        }
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            tensor_store_4d(&tmB, s_out, 0, c3_0, comp, ktl * S::P);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait<0>();
}

template <typename T>
__global__ void __launch_bounds__(kPipeThreads, Py8Smem<T>::CTAS)
k_py_inv8(const __grid_constant__ NmTensorMap tmB, typename VT<T>::V *__restrict__ A, int N3, int nTiles, int kt0,
          const typename VT<T>::V *__restrict__ wP)
{
    typedef typename VT<T>::V V;
    typedef Py8Smem<T> S;
    constexpr int M = 8;
    extern __shared__ __align__(1024) unsigned char smem[];
    V *s_in = reinterpret_cast<V *>(smem);                                  // [P][2][8]
    V *s_out = reinterpret_cast<V *>(smem + S::B_BYTES);                    // two lines, skewed
    V *s_scr = reinterpret_cast<V *>(smem + S::B_BYTES + S::A_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + S::B_BYTES + S::A_BYTES + S::SCR_BYTES);
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int h = lane & 1, l = (lane >> 1) & 1, j = lane >> 2, i = l * M + j;
    const int G = gridDim.x, H3 = N3 / 2;
    if (tid == 0) {
        mbar_init(full, 1);
        mbar_fence_init();
        tensormap_prefetch(&tmB);
    }
    __syncthreads();
    auto load_b = [&](int tl) {
        const int q = tl % H3, comp = (tl / H3) % 3, ktl = tl / (3 * H3);
        mbar_expect_tx(full, S::B_BYTES);
        tensor_load_4d(s_in, &tmB, 0, 2 * q, comp, ktl * S::P, full);
    };
    if (tid == 0 && (int)blockIdx.x < nTiles) load_b(blockIdx.x);
    V tw[16];
    load_twiddles_h<T, M>(tw, wP, j, h);
    V *scr = s_scr + (2 * w + h) * team_scratch<T, M>();
    const int coutE = l * (S::LINE_ELEMS + 2) + j * TW + (w ^ swzT<T>(j));
    const int coutO = l * (S::LINE_ELEMS + 2) + j * TW + (w ^ swzT<T>(j) ^ 4);
    int n = 0;
    for (int tl = blockIdx.x; tl < nTiles; tl += G, ++n) {
        const int c3_0 = 2 * (tl % H3);
        mbar_wait(full, (uint32_t)(n & 1));
        const int cs = w ^ swzT<T>(c3_0 + l);          // plane c3_0 + l of the pair
        V a[16];
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int u = s / M, r8 = rev8(s % M);
            const int ky = 4 * j + 2 * u + 32 * r8 + h;
            a[s] = s_in[(2 * ky + l) * TW + (cs ^ swzT<T>(4 * j + 2 * u + h))];
        }
        __syncthreads();                                    // the stage is free again
        if (tid == 0 && tl + G < nTiles) load_b(tl + G);
        fft_inv<T, M, true>(a, tw, scr, i);
        if (h) shift32<T, true>(a);
        if (tid == 0) bulk_wait_read<0>();                  // the previous tile has left s_out
        __syncthreads();
#pragma unroll
        for (int s = 0; s < 8; ++s) s_out[((s & 1) ? coutO : coutE) + M * (s + 8 * h) * TW] = half_sum(a, s, h);
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            V *dst = A + ((long long)kt0 * 3 * H3 + tl) * 2 * S::LINE_ELEMS;
            bulk_store(dst, s_out, S::LINE_ELEMS * (int)sizeof(V));
            bulk_store(dst + S::LINE_ELEMS, s_out + S::LINE_ELEMS + 2, S::LINE_ELEMS * (int)sizeof(V));
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait<0>();
}

} // namespace

// ---- host side ----------------------------------------------------------------------------------
bool nm_pipe_mid_ok(const nm_mesh *mesh)
{
    if (!mesh->fast.on || !mesh->fast.pipe) return false;
    if (mesh->f64) return (mesh->fast.M3 == 16 && mesh->fast.Kzp == Pz64Smem::KZP) || (mesh->fast.M3 == 8 && mesh->fast.Kzp == Pz64Smem8::KZP);
    if (mesh->fast.M3 == 12) return mesh->fast.Kzp == Pz3Smem::KZP;
    return (mesh->fast.M3 == 16 && mesh->fast.Kzp == PzSmem::KZP) || (mesh->fast.M3 == 8 && mesh->fast.Kzp == Pz8Smem::KZP);
}

nm_status nm_pipe_mid(nm_mesh *mesh, int kt0, int nkt, cudaStream_t st)
{
    const NmGeom &g = mesh->g;
    const int nItems = nkt * g.K2;
    const int grid = nItems < mesh->sm_count ? nItems : mesh->sm_count;
    NmLaunchScope sc(mesh, NM_K_MID, st);
    if (mesh->f64 && mesh->fast.M3 == 8) {
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Pz64Smem8::BYTES));
            kern<<<grid, kPipeThreads, Pz64Smem8::BYTES, st>>>((double2 *)mesh->bufB, (const double *)mesh->fast.Tn, mesh->fast.F2,
                                                              nItems, kt0, (const double2 *)mesh->tw_z, g.N3);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_pz_mid64_8<true>) : go(k_pz_mid64_8<false>));
        return NM_OK;
    }
    if (mesh->f64) {
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Pz64Smem::BYTES));
            kern<<<grid, kPipeThreads, Pz64Smem::BYTES, st>>>((double2 *)mesh->bufB, (const double *)mesh->fast.Tn, mesh->fast.F2,
                                                             nItems, kt0, (const double2 *)mesh->tw_z, g.N3);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_pz_mid64<true>) : go(k_pz_mid64<false>));
        return NM_OK;
    }
    if (mesh->fast.M3 == 12) {
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Pz3Smem::BYTES));
            kern<<<grid, kMidThreads, Pz3Smem::BYTES, st>>>((float2 *)mesh->bufB, (const float *)mesh->fast.Tn, mesh->fast.F2,
                                                            nItems, kt0, (const float2 *)mesh->tw_z, g.N3);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_pz_mid3<true>) : go(k_pz_mid3<false>));
        NM_CUDA_TRY(cudaGetLastError());
        return NM_OK;
    }
    if (mesh->fast.M3 == 8) {
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Pz8Smem::BYTES));
            kern<<<grid, kMidThreads, Pz8Smem::BYTES, st>>>((float2 *)mesh->bufB, (const float *)mesh->fast.Tn, mesh->fast.F2,
                                                           nItems, kt0, (const float2 *)mesh->tw_z, g.N3);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_pz_mid8<true>) : go(k_pz_mid8<false>));
        return NM_OK;
    }
    if (mesh->fast.embed) {
        NM_CUDA_TRY(cudaFuncSetAttribute(k_pz_mid<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, PzSmem::BYTES));
        k_pz_mid<true><<<grid, kMidThreads, PzSmem::BYTES, st>>>((float2 *)mesh->bufB, (const float *)mesh->fast.Tn,
                                                                 mesh->fast.F2, nItems, kt0, (const float2 *)mesh->tw_z, g.N3);
    } else {
        NM_CUDA_TRY(cudaFuncSetAttribute(k_pz_mid<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, PzSmem::BYTES));
        k_pz_mid<false><<<grid, kMidThreads, PzSmem::BYTES, st>>>((float2 *)mesh->bufB, (const float *)mesh->fast.Tn,
                                                                  mesh->fast.F2, nItems, kt0, (const float2 *)mesh->tw_z, g.N3);
    }
    return NM_OK;
}

// x passes: any fast-path size with whole CTAs of R rows along y
template <typename T, int M> nm_status launch_px(nm_mesh *mesh, bool inverse, const T *fld, T *Hc, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    typedef PxGeom<T, M> G;
    const NmGeom &g = mesh->g;
    // fewer than two CTAs per SM: one component per CTA
    const bool split = (long long)(g.N2 / G::R) * g.N3 < 2LL * mesh->sm_count;
    const dim3 grid(g.N2 / G::R, g.N3, split ? 3 : 1);
    const int f2 = mesh->fast.F2;
    if (!inverse) {
        NmLaunchScope sc(mesh, NM_K_X_FWD, st);
        auto go = [&](auto kern, T ms) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::FWD_BYTES));
            kern<<<grid, kPipeThreads, G::FWD_BYTES, st>>>(fld, (const T *)mesh->Ms, ms, (V *)mesh->bufA, g,
                                                           (const V *)mesh->fast.wPx, f2, 0);
            return NM_OK;
        };
        const T ms = (T)mesh->desc.Ms_scalar;
        if constexpr (G::BULK_OK) {
            // bulk-fed form: 16-byte aligned field, 32-bit element indices
            if (!(((uintptr_t)fld) & 15) && 3 * g.nodes < (1ll << 31) && mesh->dbg_node_path != 3) {
                const size_t bytes = G::fwd_bulk_bytes(g.n1);
                // whole grids (not split by component): persistent CTAs, two per SM, over the tiles
                const int ntiles = (int)(grid.x * grid.y);
                const int per_sm = sizeof(T) == 8 ? 1 : 2;
                const bool persist = !split && ntiles > per_sm * mesh->sm_count;
                const dim3 pgrid = persist ? dim3(per_sm * mesh->sm_count, 1, 1) : grid;
                auto gob = [&](auto kern, T msv) -> nm_status {
                    NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
                    kern<<<pgrid, kPipeThreads, bytes, st>>>(fld, (const T *)mesh->Ms, msv, (V *)mesh->bufA, g,
                                                             (const V *)mesh->fast.wPx, f2, persist ? 1 : 0);
                    return NM_OK;
                };
                if (mesh->fast.embed) NM_TRY(mesh->uni_Ms ? gob(k_px_fwd<T, M, true, true, true>, ms) : gob(k_px_fwd<T, M, false, true, true>, (T)0));
                else NM_TRY(mesh->uni_Ms ? gob(k_px_fwd<T, M, true, false, true>, ms) : gob(k_px_fwd<T, M, false, false, true>, (T)0));
                return NM_OK;
            }
        }
        if (mesh->fast.embed) NM_TRY(mesh->uni_Ms ? go(k_px_fwd<T, M, true, true, false>, ms) : go(k_px_fwd<T, M, false, true, false>, (T)0));
        else NM_TRY(mesh->uni_Ms ? go(k_px_fwd<T, M, true, false, false>, ms) : go(k_px_fwd<T, M, false, false, false>, (T)0));
    } else {
        NmLaunchScope sc(mesh, NM_K_X_INV, st);
        const int per_sm = sizeof(T) == 8 ? 1 : 2;
        const bool persist = !split && (int)(grid.x * grid.y) > per_sm * mesh->sm_count && mesh->dbg_node_path != 3;
        const dim3 pgrid = persist ? dim3(per_sm * mesh->sm_count, 1, 1) : grid;
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::INV_BYTES));
            kern<<<pgrid, kPipeThreads, G::INV_BYTES, st>>>((const V *)mesh->bufA, Hc, g, (const V *)mesh->fast.wPx, f2,
                                                            persist ? 1 : 0);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_px_inv<T, M, true>) : go(k_px_inv<T, M, false>));
    }
    return NM_OK;
}

bool nm_pipe_x_ok(const nm_mesh *mesh)
{
    if (!mesh->fast.on || !mesh->fast.pipe) return false;
    if (mesh->fast.M1 == 12) return false;                  // N1 = 192: k_fx_fwd / k_fx_inv (Len<12>)
    const int R = 2 * 8 * (16 / mesh->fast.M1);
    if (mesh->f64 && mesh->fast.M1 == 1) return false;      // the staged inverse would need more than 227 KB
    return mesh->g.N2 % R == 0;
}

template <typename T> nm_status nm_pipe_x(nm_mesh *mesh, bool inverse, const T *fld, T *Hc, cudaStream_t st)
{
    switch (mesh->fast.M1) {
    case 1: return launch_px<T, 1>(mesh, inverse, fld, Hc, st);
    case 2: return launch_px<T, 2>(mesh, inverse, fld, Hc, st);
    case 4: return launch_px<T, 4>(mesh, inverse, fld, Hc, st);
    case 8: return launch_px<T, 8>(mesh, inverse, fld, Hc, st);
    default: return launch_px<T, 16>(mesh, inverse, fld, Hc, st);
    }
}
template nm_status nm_pipe_x<float>(nm_mesh *, bool, const float *, float *, cudaStream_t);
template nm_status nm_pipe_x<double>(nm_mesh *, bool, const double *, double *, cudaStream_t);

// ---- y passes: tensor map over B and launchers ---------------------------------------------------
#include <cuda.h>

static_assert(sizeof(NmTensorMap) == sizeof(CUtensorMap), "NmTensorMap must mirror CUtensorMap");

typedef CUresult (*NmEncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// B[kt][ky][comp][c3][8 complex] seen as floats [NKT P2][3][N3][16]; box = 256 ky rows of one (comp, c3)
nm_status nm_pipe_setup(nm_mesh *mesh)
{
    mesh->fast.tmapB_ok = false;
    if (!mesh->fast.on || !mesh->fast.pipe) return NM_OK;
    const bool y8 = mesh->fast.M2 == 8 && mesh->g.N3 % 2 == 0;     // two planes per tile
    if (mesh->fast.M2 != 16 && !y8) return NM_OK;
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return NM_OK;                       // the non-pipelined y kernels serve instead
    }
    const NmGeom &g = mesh->g;
    // a row = 8 complex = 16 reals = 64 bytes (fp32) or 128 bytes (fp64)
    const cuuint64_t rowb = mesh->f64 ? 128 : 64;
    const cuuint64_t dims[4] = {16, (cuuint64_t)mesh->fast.F3, 3, (cuuint64_t)mesh->fast.NKT * g.P2};
    const cuuint64_t strides[3] = {rowb, (cuuint64_t)mesh->fast.F3 * rowb, (cuuint64_t)3 * mesh->fast.F3 * rowb};
    const cuuint32_t box[4] = {16, y8 ? 2u : 1u, 1, 256};       // M2 = 8: both planes of a tile, all 256 ky rows
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = ((NmEncodeTiledFn)fn)((CUtensorMap *)&mesh->fast.tmapB,
                                       mesh->f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, mesh->bufB,
                                       dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        nm_set_error("cuTensorMapEncodeTiled failed with code %d", (int)r);
        return NM_ECUDA;
    }
    mesh->fast.tmapB_ok = true;
    return NM_OK;
}

template <typename T> static nm_status launch_py16(nm_mesh *mesh, bool inverse, int kt0, int nkt, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    typedef PySmem<T> S;
    const NmGeom &g = mesh->g;
    const int nTiles = nkt * 3 * g.N3;
    const int cap = S::CTAS * mesh->sm_count;
    const int grid = nTiles < cap ? nTiles : cap;
    if (!inverse) {
        NmLaunchScope sc(mesh, NM_K_Y_FWD, st);
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::FWD_BYTES));
            kern<<<grid, kPipeThreads, S::FWD_BYTES, st>>>((const V *)mesh->bufA, mesh->fast.tmapB, g.N3, nTiles, kt0,
                                                           (const V *)mesh->tw_y, g.N2);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_py_fwd<T, true>) : go(k_py_fwd<T, false>));
    } else {
        NM_CUDA_TRY(cudaFuncSetAttribute(k_py_inv<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::INV_BYTES));
        NmLaunchScope sc(mesh, NM_K_Y_INV, st);
        k_py_inv<T><<<grid, kPipeThreads, S::INV_BYTES, st>>>(mesh->fast.tmapB, (V *)mesh->bufA, g.N3, nTiles, kt0,
                                                            (const V *)mesh->tw_y);
    }
    return NM_OK;
}

template <typename T> static nm_status launch_py8(nm_mesh *mesh, bool inverse, int kt0, int nkt, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    typedef Py8Smem<T> S;
    const NmGeom &g = mesh->g;
    const int nTiles = nkt * 3 * (g.N3 / 2);
    const int cap = S::CTAS * mesh->sm_count;
    const int grid = nTiles < cap ? nTiles : cap;
    if (!inverse) {
        NmLaunchScope sc(mesh, NM_K_Y_FWD, st);
        auto go = [&](auto kern) -> nm_status {
            NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, S::FWD_BYTES));
            kern<<<grid, kPipeThreads, S::FWD_BYTES, st>>>((const V *)mesh->bufA, mesh->fast.tmapB, g.N3, nTiles, kt0,
                                                           (const V *)mesh->tw_y, g.N2);
            return NM_OK;
        };
        NM_TRY(mesh->fast.embed ? go(k_py_fwd8<T, true>) : go(k_py_fwd8<T, false>));
    } else {
        NM_CUDA_TRY(cudaFuncSetAttribute(k_py_inv8<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::INV_BYTES));
        NmLaunchScope sc(mesh, NM_K_Y_INV, st);
        k_py_inv8<T><<<grid, kPipeThreads, S::INV_BYTES, st>>>(mesh->fast.tmapB, (V *)mesh->bufA, g.N3, nTiles, kt0,
                                                             (const V *)mesh->tw_y);
    }
    return NM_OK;
}

bool nm_pipe_y_ok(const nm_mesh *mesh) { return mesh->fast.on && mesh->fast.pipe && mesh->fast.tmapB_ok; }

nm_status nm_pipe_y(nm_mesh *mesh, bool inverse, int kt0, int nkt, cudaStream_t st)
{
    const NmGeom &g = mesh->g;
    if (mesh->fast.M2 == 8) return mesh->f64 ? launch_py8<double>(mesh, inverse, kt0, nkt, st) : launch_py8<float>(mesh, inverse, kt0, nkt, st);
    if (mesh->f64) return launch_py16<double>(mesh, inverse, kt0, nkt, st);
    return launch_py16<float>(mesh, inverse, kt0, nkt, st);
}
