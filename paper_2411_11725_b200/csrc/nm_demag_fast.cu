// Fast demagnetisation path: a1-a4 of the hot path for grids with N_d = 16 M_d, M_d in {1,2,4,8,16}
// (DESIGN.md "Fast demag path").  Same mathematics as nm_demag.cu (reading C5):
//   M_c = Ms_c (1/8) sum_i m_{c+i},   H_c = - sum_c' N(c - c') M_c',   P_d = 2 N_d,
// organised for B200:
//   * every transform is the register-resident radix-16 x radix-M kernel of nm_fft16.cuh; padded
//     transforms never touch their zero half,
//   * the x transform packs two real cell rows (c2, c2+1) into one complex line,
//   * spectra live in k1-blocked layouts (8 complex = 64 B per row) so that every pass moves
//     contiguous blocks:  A[kt][comp][c3][c2][8],  B[kt][ky][comp][c3][8],
//     with the 8 columns of a row XOR-swizzled by the row index of the *consuming* pass
//     (slot = k1 ^ swz(row), nm_fft16.cuh) so that its strided shared-memory reads are conflict-free,
//   * the tensor is stored as T[kt][|ky|][k1][6][|kz|] and read coalesced along kz.
// Passes: k_fx_fwd (avg * Ms, x R2C) -> k_fy_fwd -> k_fz_mid (z fwd, H^ = -N^ M^, z inv) ->
// k_fy_inv -> k_fx_inv (C2R, crop) -> Hc[3][N3][N2][N1] for the node kernel.
#include <cstdlib>

#include "nm_fft16.cuh"
#include "nm_internal.h"

using namespace nmf;

namespace {

constexpr int kWarps = 8;
constexpr int kThreadsF = 32 * kWarps;

template <typename V> __device__ __forceinline__ void copy_in(V *dst, const V *__restrict__ src, int n)
{
    // n complex elements, both 16-byte aligned, n even
    const int4 *s4 = reinterpret_cast<const int4 *>(src);
    int4 *d4 = reinterpret_cast<int4 *>(dst);
    const int n4 = n * (int)sizeof(V) / 16;
    for (int i = threadIdx.x; i < n4; i += blockDim.x) d4[i] = s4[i];
}

// -------------------------------------------------------------------------------------------------
// y forward.  CTA = LT consecutive c3 of one (kt, comp); 8 warps x LT lines.
//   in : A[kt][comp][c3][c2][8]           (rows swizzled by c2)
//   out: B[kt][ky][comp][c3][8]           (rows swizzled by c3 and ky), ky natural 0..P2-1
template <typename T, int M>
__global__ void __launch_bounds__(kThreadsF)
k_fy_fwd(const typename VT<T>::V *__restrict__ A, typename VT<T>::V *__restrict__ B, int N3, int kt0,
         const typename VT<T>::V *__restrict__ wP, int F3, int n2v)
{
    typedef typename VT<T>::V V;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    constexpr int OUT_PITCH = LT * TW + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s_io = reinterpret_cast<V *>(smem_raw);              // in: LT*N*8, out: P*OUT_PITCH
    V *s_scr = s_io + P * OUT_PITCH;                        // 2*kWarps teams
    const int c3_0 = blockIdx.x * LT;
    const int comp = blockIdx.y;
    const int kt = kt0 + blockIdx.z;
    const int ktl = blockIdx.z;                             // B is indexed relative to kt0
    const V *src = A + ((((long long)kt * 3 + comp) * N3 + c3_0) * N) * TW;
    copy_in(s_io, src, LT * N * TW);
    __syncthreads();
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = G::R3 ? min(i / MI, 2) : i / MI, j = i % MI;       // (M = 12: l = the sub-sequence, lanes with i / MI = 3 idle)
    const bool act = !G::R3 || i / MI < 3;
    const int line = G::R3 ? w : w * LT + l, sub = line / TW, k1 = line % TW;
    V tw[16];
    len_twiddles<T, M>(tw, wP, j);
    V a[16];
#pragma unroll
    for (int t = 0; t < 16; ++t) {
        const int e = len_elem<M>(l, j, t);
        V v = s_io[(sub * N + e) * TW + (k1 ^ swzT<T>(e))];
        if (e >= n2v) v = mk<T>((T)0, (T)0);                // embedded mesh: rows the x pass never wrote
        if (h) v = cmul(v, wP[len_pre<M>(l, j, t)]);
        a[t] = v;
    }
    __syncthreads();   // the input tile is dead; s_io becomes the output tile
    V *scr = s_scr + (2 * w + h) * team_scratch<T, MI>();
    len_fwd<T, M>(a, tw, scr, i, wP, lane);
    const int sl = k1 ^ swzT<T>(c3_0 + sub);
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int ky = len_freq<M>(l, j, s, h);
        if (act) s_io[ky * OUT_PITCH + sub * TW + (sl ^ swzT<T>(ky))] = a[s];
    }
    __syncthreads();
    // rows of LT*8 complex, one per ky
    V *dst = B + ((long long)ktl * P * 3 + comp) * F3 * TW + (long long)c3_0 * TW;     // B keeps F3 >= N3 planes
    for (int idx = threadIdx.x; idx < P * LT * TW; idx += blockDim.x) {
        const int ky = idx / (LT * TW), r = idx % (LT * TW);
        dst[(long long)ky * 3 * F3 * TW + r] = s_io[ky * OUT_PITCH + r];
    }
}

// y inverse, cropped to N2.  in: B (as above), out: A layout (rows swizzled by c2).
template <typename T, int M>
__global__ void __launch_bounds__(kThreadsF)
k_fy_inv(const typename VT<T>::V *__restrict__ B, typename VT<T>::V *__restrict__ A, int N3, int kt0,
         const typename VT<T>::V *__restrict__ wP, int F3)
{
    typedef typename VT<T>::V V;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    constexpr int PITCH = LT * TW + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s_io = reinterpret_cast<V *>(smem_raw);              // in: P*PITCH, out: LT*N*8
    V *s_scr = s_io + P * PITCH;
    const int c3_0 = blockIdx.x * LT;
    const int comp = blockIdx.y;
    const int kt = kt0 + blockIdx.z;
    const int ktl = blockIdx.z;
    const V *src = B + ((long long)ktl * P * 3 + comp) * F3 * TW + (long long)c3_0 * TW;
    for (int idx = threadIdx.x; idx < P * LT * TW; idx += blockDim.x) {
        const int ky = idx / (LT * TW), r = idx % (LT * TW);
        s_io[ky * PITCH + r] = src[(long long)ky * 3 * F3 * TW + r];
    }
    __syncthreads();
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = G::R3 ? min(i / MI, 2) : i / MI, j = i % MI;       // (M = 12: l = the sub-sequence, lanes with i / MI = 3 idle)
    const bool act = !G::R3 || i / MI < 3;
    const int line = G::R3 ? w : w * LT + l, sub = line / TW, k1 = line % TW;
    V tw[16];
    len_twiddles<T, M>(tw, wP, j);
    V a[16];
    const int sl = k1 ^ swzT<T>(c3_0 + sub);
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int ky = len_freq<M>(l, j, s, h);
        a[s] = s_io[ky * PITCH + sub * TW + (sl ^ swzT<T>(ky))];
    }
    __syncthreads();
    V *scr = s_scr + (2 * w + h) * team_scratch<T, MI>();
    len_inv<T, M>(a, tw, scr, i, wP, lane);
#pragma unroll
    for (int t = 0; t < 16; ++t) {
        const int e = len_elem<M>(l, j, t);
        V v = a[t];
        if (h) v = cmulc(v, wP[len_pre<M>(l, j, t)]);
        // sum of the even and odd halves: partner lane = lane ^ 1
        v = cadd(v, shfl1(v));
        if ((t >> 3) == h && act) s_io[(sub * N + e) * TW + (k1 ^ swzT<T>(e))] = v;
    }
    __syncthreads();
    V *dst = A + ((((long long)kt * 3 + comp) * N3 + c3_0) * N) * TW;
    copy_in(dst, s_io, LT * N * TW);
}

// -------------------------------------------------------------------------------------------------
// z forward, tensor multiply, z inverse, in place on B.  CTA = LT consecutive ky of one kt.
//   Tn[kt][|ky|][k1][6][|kz|] (pitch Kzp), components xx,yy,zz,xy,xz,yz, scaled by 1/(P1 P2 P3);
//   off-diagonal components are odd in their two axes: sign -1 per folded axis (ky > N2, kz > N3).
template <typename T, int M, bool EMB>
__global__ void __launch_bounds__(kThreadsF)
k_fz_mid(typename VT<T>::V *__restrict__ B, const T *__restrict__ Tn, int N2, int kt0, int Kzp,
         const typename VT<T>::V *__restrict__ wP, int n3v)
{
    typedef typename VT<T>::V V;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s_io = reinterpret_cast<V *>(smem_raw);              // LT*3*N*8
    V *s_scr = s_io + LT * 3 * N * TW;
    const int P2 = 2 * N2;
    int ky0;
    if (LT == 1) {
        // +ky and -ky in neighbouring CTAs: they read the same folded tensor rows
        const int it = blockIdx.x;
        ky0 = (it & 1) ? P2 - ((it + 1) >> 1) : (it >> 1);
    } else {
        ky0 = blockIdx.x * LT;
    }
    const int ktl = blockIdx.y, kt = kt0 + ktl;
    V *tile = B + (((long long)ktl * P2 + ky0) * 3 * N) * TW;
    copy_in(s_io, tile, LT * 3 * N * TW);
    __syncthreads();
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = G::R3 ? min(i / MI, 2) : i / MI, j = i % MI;       // (M = 12: l = the sub-sequence, lanes with i / MI = 3 idle)
    const bool act = !G::R3 || i / MI < 3;
    const int line = G::R3 ? w : w * LT + l, sub = line / TW, k1 = line % TW;
    V *scr = s_scr + (2 * w + h) * team_scratch<T, MI>();
    V tw[16];
    len_twiddles<T, M>(tw, wP, j);
    V a[3][16];
    V *my = s_io + (sub * 3) * N * TW;
    const int kq = k1 ^ swzT<T>(ky0 + sub);                     // rows of B are swizzled by c3 and by ky
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const int e = len_elem<M>(l, j, t);
            V v = my[(c * N + e) * TW + (kq ^ swzT<T>(e))];
            if (EMB && e >= n3v) v = mk<T>((T)0, (T)0);     // embedded mesh: planes the y pass never wrote
            if (h) v = cmul(v, wP[len_pre<M>(l, j, t)]);
            a[c][t] = v;
        }
        len_fwd<T, M>(a[c], tw, scr, i, wP, lane);
    }
    // H^ = -N^ M^
    const int ky = ky0 + sub;
    const int kyf = ky <= N2 ? ky : P2 - ky;
    const T sy = ky <= N2 ? (T)1 : (T)-1;
    const long long cstride = Kzp;
    const T *trow = Tn + ((((long long)kt * (N2 + 1) + kyf) * TW + k1) * 6) * Kzp;
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int kz = len_freq<M>(l, j, s, h);
        const int kzf = kz <= N ? kz : P - kz;
        const T sz = kz <= N ? (T)1 : (T)-1;
        const T *tp = trow + kzf;
        const T nxx = tp[0], nyy = tp[cstride], nzz = tp[2 * cstride];
        const T nxy = sy * tp[3 * cstride], nxz = sz * tp[4 * cstride], nyz = sy * sz * tp[5 * cstride];
        const V mx = a[0][s], my_ = a[1][s], mz = a[2][s];
        const V hx = caxpy(nxz, mz, caxpy(nxy, my_, cscale(nxx, mx)));
        const V hy = caxpy(nyz, mz, caxpy(nyy, my_, cscale(nxy, mx)));
        const V hz = caxpy(nzz, mz, caxpy(nyz, my_, cscale(nxz, mx)));
        a[0][s] = mk<T>(-hx.x, -hx.y);
        a[1][s] = mk<T>(-hy.x, -hy.y);
        a[2][s] = mk<T>(-hz.x, -hz.y);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        len_inv<T, M>(a[c], tw, scr, i, wP, lane);
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const int e = len_elem<M>(l, j, t);
            V v = a[c][t];
            if (h) v = cmulc(v, wP[len_pre<M>(l, j, t)]);
            v = cadd(v, shfl1(v));
            if ((t >> 3) == h && act) my[(c * N + e) * TW + (kq ^ swzT<T>(e))] = v;
        }
    }
    __syncthreads();
    copy_in(tile, s_io, LT * 3 * N * TW);
}

// -------------------------------------------------------------------------------------------------
// x forward: node -> cell average times Ms (a1), two real cell rows (c2, c2+1) per complex line,
// padded transform, untangle, blocked store.  CTA = R = 2 LT W cell rows of one c3, all components.
template <typename T, int M>
__global__ void __launch_bounds__(kThreadsF)
k_fx_fwd(const T *__restrict__ fld, const T *__restrict__ Ms, typename VT<T>::V *__restrict__ A, NmGeom g,
         int NKT, const typename VT<T>::V *__restrict__ wP)
{
    typedef typename VT<T>::V V;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    const int W = blockDim.x >> 5;
    const int R = 2 * LT * W;
    constexpr int CP = N + 1;                               // cell row pitch (reals)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s_z = reinterpret_cast<V *>(smem_raw);               // W*LT lines x P
    V *s_scr = s_z + W * LT * P;                            // 2 W teams
    T *s_cell = reinterpret_cast<T *>(s_scr + 2 * W * team_scratch<T, MI>());   // R x CP
    const int r0 = blockIdx.x * R, c3 = blockIdx.y;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = G::R3 ? min(i / MI, 2) : i / MI, j = i % MI;
    const bool act = !G::R3 || i / MI < 3;
    const int line = G::R3 ? w : w * LT + l;
    V *scr = s_scr + (2 * w + h) * team_scratch<T, MI>();
    V tw[16];
    len_twiddles<T, M>(tw, wP, j);
    const long long plane = (long long)g.n1 * g.n2;
    // small grids: one component per CTA (gridDim.z = 3)
    for (int comp = gridDim.z == 3 ? (int)blockIdx.z : 0; comp < (gridDim.z == 3 ? (int)blockIdx.z + 1 : 3); ++comp) {
        // a1: M_c = Ms_c (1/8) sum of the 8 vertices
        const T *base = fld + (long long)comp * g.nodes + (long long)c3 * plane;
        for (int idx = threadIdx.x; idx < R * N; idx += blockDim.x) {
            const int r = idx / N, c1 = idx % N;
            const int c2 = r0 + r;
            const T *p = base + (long long)c2 * g.n1 + c1;
            const T sum = ((p[0] + p[1]) + (p[g.n1] + p[g.n1 + 1])) +
                          ((p[plane] + p[plane + 1]) + (p[plane + g.n1] + p[plane + g.n1 + 1]));
            s_cell[r * CP + c1] = Ms[((long long)c3 * g.N2 + c2) * g.N1 + c1] * (T)0.125 * sum;
        }
        __syncthreads();
        V a[16];
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const int e = len_elem<M>(l, j, t);
            V v = mk<T>(s_cell[(2 * line) * CP + e], s_cell[(2 * line + 1) * CP + e]);
            if (h) v = cmul(v, wP[len_pre<M>(l, j, t)]);
            a[t] = v;
        }
        len_fwd<T, M>(a, tw, scr, i, wP, lane);
#pragma unroll
        for (int s = 0; s < 16; ++s)
            if (act) s_z[line * P + len_freq<M>(l, j, s, h)] = a[s];
        __syncthreads();
        // untangle the two real rows of each line and store blocked, swizzled by c2
        for (int idx = threadIdx.x; idx < NKT * R * TW; idx += blockDim.x) {
            const int kt = idx / (R * TW), rem = idx % (R * TW);
            const int r = rem / TW, slot = rem % TW;
            const int c2 = r0 + r;
            const int k = kt * TW + (slot ^ swzT<T>(c2));
            V out = mk<T>((T)0, (T)0);
            if (k <= N) {
                const V zk = s_z[(r >> 1) * P + k];
                const V zm = s_z[(r >> 1) * P + (k ? P - k : 0)];
                if (r & 1) out = mk<T>((T)0.5 * (zk.y + zm.y), (T)-0.5 * (zk.x - zm.x));
                else out = mk<T>((T)0.5 * (zk.x + zm.x), (T)0.5 * (zk.y - zm.y));
            }
            A[((((long long)kt * 3 + comp) * g.N3 + c3) * g.N2 + r0) * TW + rem] = out;
        }
        __syncthreads();
    }
}

// x inverse: rebuild the packed spectrum of two real rows from their half spectra, inverse
// transform cropped to N1, write the cell field Hc[comp][c3][c2][c1].
template <typename T, int M>
__global__ void __launch_bounds__(kThreadsF)
k_fx_inv(const typename VT<T>::V *__restrict__ A, T *__restrict__ Hc, NmGeom g, int NKT,
         const typename VT<T>::V *__restrict__ wP)
{
    typedef typename VT<T>::V V;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    const int W = blockDim.x >> 5;
    const int R = 2 * LT * W;
    const int XP = NKT * TW + 1;                            // row pitch of s_x (complex)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s_x = reinterpret_cast<V *>(smem_raw);               // R x XP
    V *s_scr = s_x + R * XP;
    const int r0 = blockIdx.x * R, c3 = blockIdx.y;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane & 1, i = lane >> 1;
    const int l = G::R3 ? min(i / MI, 2) : i / MI, j = i % MI;
    const bool act = !G::R3 || i / MI < 3;
    const int line = G::R3 ? w : w * LT + l;
    V *scr = s_scr + (2 * w + h) * team_scratch<T, MI>();
    V tw[16];
    len_twiddles<T, M>(tw, wP, j);
    // small grids: one component per CTA (gridDim.z = 3)
    for (int comp = gridDim.z == 3 ? (int)blockIdx.z : 0; comp < (gridDim.z == 3 ? (int)blockIdx.z + 1 : 3); ++comp) {
        for (int idx = threadIdx.x; idx < NKT * R * TW; idx += blockDim.x) {
            const int kt = idx / (R * TW), rem = idx % (R * TW);
            const int r = rem / TW, slot = rem % TW;
            const int c2 = r0 + r;
            s_x[r * XP + kt * TW + (slot ^ swzT<T>(c2))] =
                A[((((long long)kt * 3 + comp) * g.N3 + c3) * g.N2 + r0) * TW + rem];
        }
        __syncthreads();
        V a[16];
        const V *xa = s_x + (2 * line) * XP, *xb = xa + XP;
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int k = len_freq<M>(l, j, s, h);
            if (k <= N) {
                const V u = xa[k], v = xb[k];
                a[s] = mk<T>(u.x - v.y, u.y + v.x);          // Xa + i Xb
            } else {
                const V u = xa[P - k], v = xb[P - k];
                a[s] = mk<T>(u.x + v.y, v.x - u.y);          // conj(Xa) + i conj(Xb)
            }
        }
        len_inv<T, M>(a, tw, scr, i, wP, lane);
        T *ha = Hc + (long long)comp * g.cells + ((long long)c3 * g.N2 + r0 + 2 * line) * g.N1;
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const int e = len_elem<M>(l, j, t);
            V v = a[t];
            if (h) v = cmulc(v, wP[len_pre<M>(l, j, t)]);
            v = cadd(v, shfl1(v));
            if ((t >> 3) == h && act) {
                ha[e] = v.x;
                ha[g.N1 + e] = v.y;
            }
        }
        __syncthreads();
    }
}

template <typename K> nm_status set_smem_f(K kernel, size_t bytes)
{
    if (bytes > 48 * 1024)
        NM_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return NM_OK;
}

template <typename T> size_t scratch_bytes(int warps)
{
    return (size_t)2 * warps * team_scratch<T, 16>() * sizeof(typename VT<T>::V);
}

// ---- per-axis launchers (M is a template parameter of the kernels) ----
template <typename T, int M>
nm_status launch_x(nm_mesh *mesh, bool inverse, const T *fld, T *Hc, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    const NmGeom &g = mesh->g;
    const NmFast &f = mesh->fast;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    const int W = f.Wx, R = 2 * LT * W;
    const bool split = (long long)(g.N2 / R) * g.N3 < 2LL * mesh->sm_count;
    const dim3 grid(g.N2 / R, g.N3, split ? 3 : 1);
    if (!inverse) {
        const size_t sm = (size_t)W * LT * P * sizeof(V) + scratch_bytes<T>(W) + (size_t)R * (N + 1) * sizeof(T);
        NM_TRY(set_smem_f(k_fx_fwd<T, M>, sm));
        NmLaunchScope sc(mesh, NM_K_X_FWD, st);
        k_fx_fwd<T, M><<<grid, 32 * W, sm, st>>>(fld, (const T *)mesh->Ms, (V *)mesh->bufA, g, f.NKT,
                                                 (const V *)f.wPx);
    } else {
        const size_t sm = (size_t)R * (f.NKT * TW + 1) * sizeof(V) + scratch_bytes<T>(W);
        NM_TRY(set_smem_f(k_fx_inv<T, M>, sm));
        NmLaunchScope sc(mesh, NM_K_X_INV, st);
        k_fx_inv<T, M><<<grid, 32 * W, sm, st>>>((const V *)mesh->bufA, Hc, g, f.NKT, (const V *)f.wPx);
    }
    return NM_OK;
}

template <typename T, int M>
nm_status launch_y(nm_mesh *mesh, bool inverse, int kt0, int nkt, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    const NmGeom &g = mesh->g;
    typedef Len<M> G;
    constexpr int N = G::N, P = G::P, LT = G::LT, MI = G::MI;
    if (nm_pipe_y_ok(mesh)) return nm_pipe_y(mesh, inverse, kt0, nkt, st);
    const size_t sm = (size_t)P * (LT * TW + 1) * sizeof(V) + scratch_bytes<T>(kWarps);
    const dim3 grid(g.N3 / LT, 3, nkt);
    if (!inverse) {
        NM_TRY(set_smem_f(k_fy_fwd<T, M>, sm));
        NmLaunchScope sc(mesh, NM_K_Y_FWD, st);
        k_fy_fwd<T, M><<<grid, kThreadsF, sm, st>>>((const V *)mesh->bufA, (V *)mesh->bufB, g.N3, kt0,
                                                    (const V *)mesh->tw_y, mesh->fast.F3, g.N2);
    } else {
        NM_TRY(set_smem_f(k_fy_inv<T, M>, sm));
        NmLaunchScope sc(mesh, NM_K_Y_INV, st);
        k_fy_inv<T, M><<<grid, kThreadsF, sm, st>>>((const V *)mesh->bufB, (V *)mesh->bufA, g.N3, kt0,
                                                    (const V *)mesh->tw_y, mesh->fast.F3);
    }
    return NM_OK;
}

template <typename T, int M>
nm_status launch_z(nm_mesh *mesh, int kt0, int nkt, cudaStream_t st)
{
    typedef typename VT<T>::V V;
    const NmGeom &g = mesh->g;
    typedef Len<M> G;
    constexpr int N = G::N, LT = G::LT;
    if (nm_pipe_mid_ok(mesh)) return nm_pipe_mid(mesh, kt0, nkt, st);
    const size_t sm = (size_t)LT * 3 * N * TW * sizeof(V) + scratch_bytes<T>(kWarps);
    const dim3 grid(g.P2 / LT, nkt);
    NmLaunchScope sc(mesh, NM_K_MID, st);
    if (mesh->fast.embed) {
        NM_TRY(set_smem_f(k_fz_mid<T, M, true>, sm));
        k_fz_mid<T, M, true><<<grid, kThreadsF, sm, st>>>((V *)mesh->bufB, (const T *)mesh->fast.Tn, mesh->fast.F2, kt0,
                                                          mesh->fast.Kzp, (const V *)mesh->tw_z, g.N3);
    } else {
        NM_TRY(set_smem_f(k_fz_mid<T, M, false>, sm));
        k_fz_mid<T, M, false><<<grid, kThreadsF, sm, st>>>((V *)mesh->bufB, (const T *)mesh->fast.Tn, mesh->fast.F2, kt0,
                                                           mesh->fast.Kzp, (const V *)mesh->tw_z, g.N3);
    }
    return NM_OK;
}

#define NM_SWITCH_M(Mv, CALL)                                                                          \
    switch (Mv) {                                                                                      \
    case 1: { constexpr int MM = 1; NM_TRY(CALL); } break;                                             \
    case 2: { constexpr int MM = 2; NM_TRY(CALL); } break;                                             \
    case 4: { constexpr int MM = 4; NM_TRY(CALL); } break;                                             \
    case 8: { constexpr int MM = 8; NM_TRY(CALL); } break;                                             \
    case 12: { constexpr int MM = 12; NM_TRY(CALL); } break;                                           \
    default: { constexpr int MM = 16; NM_TRY(CALL); } break;                                           \
    }

// tensor in the fast layout from the folded fp64 octant in[6][K3][K2][K1]
template <typename T>
__global__ void k_tensor_store_fast(const double *__restrict__ in, T *__restrict__ Tn, int K1, int K2,
                                    int K3, int NKT, int Kzp, double scale)
{
    const long long total = (long long)NKT * K2 * 6 * TW * Kzp;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    long long r = idx;
    const int kz = (int)(r % Kzp); r /= Kzp;
    const int a = (int)(r % 6); r /= 6;
    const int k1 = (int)(r % TW); r /= TW;
    const int ky = (int)(r % K2);
    const int kt = (int)(r / K2);
    const int kx = kt * TW + k1;
    double v = 0.0;
    if (kx < K1 && kz < K3) {
        v = in[(((long long)a * K3 + kz) * K2 + ky) * K1 + kx] * scale;
        if (a >= 3) v = -v;   // (-i)^2 from the two odd axes
    }
    Tn[idx] = (T)v;
}

} // namespace

// Which grids the fast path serves, and its sizes.  Host only.
// Exact sizes: every N_d in {16,...,256}.  Embedded sizes: any 2 <= N_d <= 256 that fills at least
// half of the (y, z) plane of the next fast sizes F_d and meets the CTA granularities below -- the
// convolution is then computed on the zero-extended 2 F_d grid
// (longer than the 2 N_d - 1 a linear convolution needs, so the result is the same), the x passes
// touching only the N1 x N2 x N3 cells that exist and the y / z passes masking the rows that do not.
void nm_fast_plan(const nm_mesh_desc *d, const NmGeom &g, NmFast *f)
{
    f->on = false;
    f->embed = false;
    if (!(d->terms & NM_TERM_DEMAG)) return;
    int M[3], F[3];
    const int N[3] = {g.N1, g.N2, g.N3};
    // NM_FAST192=1 (read at nm_mesh_create): an axis of 192 cells is transformed at its own length (Len<12>, nm_fft16.cuh:
    // 192 = 3 x 64) instead of zero-extended to 256.  Off by default: measured slower (profiles/r2_final.md) -- the
    // 192-cell forms exist for the one-CTA-per-tile kernels k_fx_* / k_fy_* and for the z pass (k_pz_mid3) only, and
    // the persistent pipelines at 256 cells make up for 2.4 times the work.
    const char *e192 = getenv("NM_FAST192");
    const bool native192 = e192 && e192[0] == '1';
    bool exact = true;
    for (int a = 0; a < 3; ++a) {
        if (N[a] > 256) return;
        F[a] = 16;
        while (F[a] < N[a]) F[a] *= 2;
        if (N[a] == 192 && native192) F[a] = 192;    // 3 x 64: the radix-3 form of the register core (Len<12>)
        if (F[a] != N[a]) exact = false;
        M[a] = F[a] / 16;
    }
    if (!exact)                                      // embedded meshes know the sizes 16 * 2^k only
        for (int a = 0; a < 3; ++a)
            if (F[a] == 192) { F[a] = 256; M[a] = 16; }
    const int LTx = M[0] == 12 ? 1 : 16 / M[0];
    if (!exact) {
        const int vec = d->dtype == NM_F64 ? 2 : 4;
        if (N[0] < 2 || N[1] < 2 || N[2] < 2) return;                           // films and rods: the 2-D / 1-D general path
        // a mesh the general path can serve (every N_d = 2^a 3^b) is embedded only where that is faster:
        // it must fill 1/2 (pipelined y / z kernels) or 3/4 of the (y, z) plane the z pass transforms in full
        bool smooth = true;
        for (int a = 0; a < 3; ++a) {
            int v = N[a];
            while (v % 2 == 0) v /= 2;
            while (v % 3 == 0) v /= 3;
            if (v != 1) smooth = false;
        }
        const long long fill = (long long)N[1] * N[2] * 4, plane = (long long)F[1] * F[2];
        // (fp64 has pipelined y / z kernels at 128 and 256 cells only: smaller extended planes must be fuller to pay)
        const bool piped = d->dtype != NM_F64 || ((F[1] == 256 || F[1] == 128) && (F[2] == 256 || F[2] == 128));
        if (smooth && fill < (piped ? 2 : 3) * plane) return;
        if (N[1] % (2 * 8 * LTx) != 0 || N[0] % vec != 0) return;              // whole x-pass CTAs of rows, 16-byte cell rows
        if (N[2] % (16 / M[1]) != 0) return;                                   // whole y-pass CTAs of planes (M = 12 never gets here)
        if (d->dtype == NM_F64 && M[0] == 1) return;                           // no staged fp64 x pass at N1 = 16
        f->embed = true;
    }
    int W = kWarps;
    while (W >= 1 && (N[1] % (2 * LTx * W)) != 0) W >>= 1;
    if (W < 1) return;
    f->M1 = M[0]; f->M2 = M[1]; f->M3 = M[2];
    f->F1 = F[0]; f->F2 = F[1]; f->F3 = F[2];
    f->Wx = W;
    f->NKT = (F[0] + 1 + TW - 1) / TW;
    f->Kzp = (F[2] + 1 + 1) & ~1;   // even: a warp's 6 rows are a multiple of 16 bytes
    f->on = true;
}

// (g here already carries the transform extents in P_d, C1, K_d)
size_t nm_fast_tensor_elems(const NmGeom &g, const NmFast &f)
{
    return (size_t)f.NKT * g.K2 * 6 * TW * f.Kzp;
}
// A[kt][comp][c3 < N3][c2 < F2][8], B[kt][ky < 2 F2][comp][c3 < F3][8]
size_t nm_fast_bufA_elems(const NmGeom &g, const NmFast &f) { return (size_t)f.NKT * 3 * g.N3 * f.F2 * TW; }
size_t nm_fast_bufB_elems(const NmGeom &g, const NmFast &f) { return (size_t)f.NKT * g.P2 * 3 * f.F3 * TW; }

nm_status nm_fast_store_tensor(nm_mesh *mesh, const double *octant, double scale, cudaStream_t st)
{
    const NmGeom &g = mesh->g;
    const NmFast &f = mesh->fast;
    const long long total = (long long)nm_fast_tensor_elems(g, f);
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (mesh->f64)
        k_tensor_store_fast<double><<<blocks, 256, 0, st>>>(octant, (double *)f.Tn, g.C1, g.K2, g.K3, f.NKT, f.Kzp, scale);
    else
        k_tensor_store_fast<float><<<blocks, 256, 0, st>>>(octant, (float *)f.Tn, g.C1, g.K2, g.K3, f.NKT, f.Kzp, scale);
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T>
nm_status nm_demag_conv_fast(nm_mesh *mesh, const T *fld, T *Hc_out, cudaStream_t st)
{
    const NmFast &f = mesh->fast;
    const bool px = nm_pipe_x_ok(mesh);
    if (px) NM_TRY(nm_pipe_x<T>(mesh, false, fld, Hc_out, st));
    else NM_SWITCH_M(f.M1, (launch_x<T, MM>(mesh, false, fld, Hc_out, st)));
    const int chunk = f.kt_chunk > 0 && f.kt_chunk < f.NKT ? f.kt_chunk : f.NKT;
    for (int kt0 = 0; kt0 < f.NKT; kt0 += chunk) {
        const int nkt = kt0 + chunk <= f.NKT ? chunk : f.NKT - kt0;
        NM_SWITCH_M(f.M2, (launch_y<T, MM>(mesh, false, kt0, nkt, st)));
        NM_SWITCH_M(f.M3, (launch_z<T, MM>(mesh, kt0, nkt, st)));
        NM_SWITCH_M(f.M2, (launch_y<T, MM>(mesh, true, kt0, nkt, st)));
    }
    if (px) NM_TRY(nm_pipe_x<T>(mesh, true, fld, Hc_out, st));
    else NM_SWITCH_M(f.M1, (launch_x<T, MM>(mesh, true, fld, Hc_out, st)));
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template nm_status nm_demag_conv_fast<float>(nm_mesh *, const float *, float *, cudaStream_t);
template nm_status nm_demag_conv_fast<double>(nm_mesh *, const double *, double *, cudaStream_t);
