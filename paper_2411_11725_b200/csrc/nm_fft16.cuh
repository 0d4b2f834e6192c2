// Register-resident FFT core of the fast demag path (device code).
//
// a2/a4 of the hot path: zero-padded transforms of the demag convolution
// (PAPER.md:175-181).  A padded transform of length P = 2N whose upper input half is zero splits
// exactly into two N-point transforms,
//     X[2k]   = FFT_N(x)[k],            X[2k+1] = FFT_N(x[n] w_P^n)[k],         w_P = exp(-2 pi i/P)
// and the cropped inverse into
//     y[n]    = IFFT_N(X_even)[n] + conj(w_P^n) IFFT_N(X_odd)[n],   n < N,
// so no thread ever touches the zero half.  N = 16 M, M in {1,2,4,8,16}.  A *team* of 16 threads
// holds 16 complex values each and transforms 16/M lines at once:
//     stage 1   radix-16 butterfly over the register index t (elements j + M t of a line)
//     twiddle   w_N^(j t')
//     exchange  through a team-private, conflict-free shared-memory scratch (warp-synchronous)
//     stage 2   radix-M butterflies
// The spectrum stays in the scrambled register order stage 2 leaves it in (slot_freq below); the
// inverse runs the same steps backwards, so no reordering pass exists.  Two teams share a warp:
// lane = 2 i + h, team h = 0 takes the even outputs, h = 1 the odd ones.
#pragma once

#include "nm_internal.h"
#include "nm_pair.cuh"

namespace nmf {

using namespace nmp;

template <typename T> struct VT { typedef typename NmVec2<T>::type V; };

constexpr int TW = 8;   // complex columns (k1) per blocked spectrum row

// Column swizzle of a blocked row: the 8 columns of row r (r = the index the consuming pass
// transforms along) are stored at slot = k1 ^ swz(r).  16 consecutive rows of one column then
// fall into 16 different 8-byte bank pairs of shared memory (row parity picks the half, swz the
// slot), so the strided column reads of the consuming pass are conflict-free.
__host__ __device__ __forceinline__ int swz(int r) { return (r >> 1) & 7; }
// The swizzle by precision.  fp64 elements are 16 bytes and a row of 8 is the whole 128-byte bank period, so
// which banks an access uses is the slot alone, and a 128-bit access is served eight lanes at a time: the rows
// one such group touches -- four consecutive rows of a column (both halves of a team read the same element),
// or eight consecutive rows where the halves own alternate rows -- must sit in different slots.  Row parity,
// which picks the bank half in fp32, therefore goes into the slot: 8 consecutive rows -> slots 0,4,1,5,2,6,3,7.
template <typename T> __host__ __device__ __forceinline__ int swzT(int r)
{
    return sizeof(T) == 8 ? (((r >> 1) & 7) ^ ((r & 1) << 2)) : ((r >> 1) & 7);
}

template <typename T> __device__ __forceinline__ typename VT<T>::V mk(T a, T b)
{
    typename VT<T>::V v;
    v.x = a;
    v.y = b;
    return v;
}
template <typename V> __device__ __forceinline__ V cadd(V a, V b) { a.x += b.x; a.y += b.y; return a; }
template <typename V> __device__ __forceinline__ V csub(V a, V b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename V> __device__ __forceinline__ V cmul(V a, V b)
{
    V r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
template <typename V> __device__ __forceinline__ V cmulc(V a, V b)   // a * conj(b)
{
    V r;
    r.x = a.x * b.x + a.y * b.y;
    r.y = a.y * b.x - a.x * b.y;
    return r;
}
// fp32 complex arithmetic on packed pairs (nm_pair.cuh); these non-template overloads win over the
// templates above for float2 arguments
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return padd(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return psub(a, b); }
__device__ __forceinline__ float2 cmul(float2 a, float2 w)     // (ax wx - ay wy, ax wy + ay wx)
{
    const float2 t = pmul(make_float2(a.y, a.y), make_float2(w.y, w.x));
    return pfma(make_float2(a.x, a.x), w, make_float2(-t.x, t.y));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 w)    // (ax wx + ay wy, ay wx - ax wy)
{
    const float2 t = pmul(make_float2(a.x, a.x), w);
    return pfma(make_float2(a.y, a.y), make_float2(w.y, w.x), make_float2(t.x, -t.y));
}
// a * (c - i s): forward twiddle with compile-time c, s (INV: a * (c + i s)); the constants ride as
// broadcast immediates
template <bool INV> __device__ __forceinline__ float2 cmul_cs(float2 a, float c, float s)
{
    const float2 t = pmul(make_float2(a.y, a.x), make_float2(s, s));        // (s ay, s ax)
    return pfma(a, make_float2(c, c), INV ? make_float2(-t.x, t.y) : make_float2(t.x, -t.y));
}
template <bool INV> __device__ __forceinline__ double2 cmul_cs(double2 a, double c, double s)
{
    double2 r;
    if (INV) { r.x = a.x * c - a.y * s; r.y = a.y * c + a.x * s; }
    else { r.x = a.x * c + a.y * s; r.y = a.y * c - a.x * s; }
    return r;
}
// s * a and a + s * b with a real scalar s
__device__ __forceinline__ float2 cscale(float s, float2 a) { return pmul(a, make_float2(s, s)); }
__device__ __forceinline__ float2 caxpy(float s, float2 b, float2 a) { return pfma(b, make_float2(s, s), a); }
__device__ __forceinline__ double2 cscale(double s, double2 a) { a.x *= s; a.y *= s; return a; }
__device__ __forceinline__ double2 caxpy(double s, double2 b, double2 a) { a.x += s * b.x; a.y += s * b.y; return a; }

// the value held by the partner lane (lane ^ 1: the other half h of the same team thread)
template <typename V> __device__ __forceinline__ V shfl1(V v)
{
    V r;
    r.x = __shfl_xor_sync(0xffffffffu, v.x, 1);
    r.y = __shfl_xor_sync(0xffffffffu, v.y, 1);
    return r;
}

// Sum of the even and odd halves of output row t = s + 8 h (s = 0..7) of an inverse padded transform: the lane of half
// h keeps the rows t = s + 8 h, sends its partner the value the partner keeps and adds the one it receives -- one
// exchange per kept value (adding the halves of all 16 rows on both lanes and dropping eight costs two).
template <typename V> __device__ __forceinline__ V half_sum(const V *a, int s, int h)
{
    const V give = h ? a[s] : a[s + 8], keep = h ? a[s + 8] : a[s];
    return cadd(keep, shfl1(give));
}

// a * w (INV = false) or a * conj(w) (INV = true)
template <bool INV, typename V> __device__ __forceinline__ V ctw(V a, V w)
{
    return INV ? cmulc(a, w) : cmul(a, w);
}
// multiply by -i (forward) / +i (inverse)
template <bool INV, typename V> __device__ __forceinline__ V rot90(V a)
{
    V r;
    if (INV) { r.x = -a.y; r.y = a.x; }
    else { r.x = a.y; r.y = -a.x; }
    return r;
}

// 4-point DFT, natural order in and out; sign -1 (forward) or +1 (INV).
template <bool INV, typename V> __device__ __forceinline__ void dft4(V &a0, V &a1, V &a2, V &a3)
{
    const V s02 = cadd(a0, a2), d02 = csub(a0, a2);
    const V s13 = cadd(a1, a3), d13 = rot90<INV>(csub(a1, a3));
    a0 = cadd(s02, s13);
    a2 = csub(s02, s13);
    a1 = cadd(d02, d13);
    a3 = csub(d02, d13);
}

template <typename V> __device__ __forceinline__ void dft2(V &a0, V &a1)
{
    const V s = cadd(a0, a1), d = csub(a0, a1);
    a0 = s;
    a1 = d;
}

// exp(-+ 2 pi i q/16) as compile-time constants
template <typename T, bool INV, int Q> __device__ __forceinline__ typename VT<T>::V mul_w16(typename VT<T>::V a)
{
    typedef typename VT<T>::V V;
    constexpr int q = ((Q % 16) + 16) % 16;
    const T c1 = (T)0.92387953251128675612818318939679;   // cos(pi/8)
    const T s1 = (T)0.38268343236508977172845998403040;   // sin(pi/8)
    const T h = (T)0.70710678118654752440084436210485;
    if (q == 0) return a;
    if (q == 4) return rot90<INV>(a);
    if (q == 8) return mk<T>(-a.x, -a.y);
    if (q == 12) return rot90<!INV>(a);
    T c, s;   // w = c - i s (forward)
    if (q == 1) { c = c1; s = s1; }
    else if (q == 2) { c = h; s = h; }
    else if (q == 3) { c = s1; s = c1; }
    else if (q == 5) { c = -s1; s = c1; }
    else if (q == 6) { c = -h; s = h; }
    else if (q == 7) { c = -c1; s = s1; }
    else if (q == 9) { c = -c1; s = -s1; }
    else if (q == 10) { c = -h; s = -h; }
    else if (q == 11) { c = -s1; s = -c1; }
    else if (q == 13) { c = s1; s = -c1; }
    else if (q == 14) { c = h; s = -h; }
    else { c = c1; s = -s1; }   // 15
    return cmul_cs<INV>(a, c, s);
}

// exp(-+ 2 pi i q/32) as compile-time constants, q = 0..15
template <typename T, bool INV, int Q> __device__ __forceinline__ typename VT<T>::V mul_w32(typename VT<T>::V a)
{
    typedef typename VT<T>::V V;
    if (Q % 2 == 0) return mul_w16<T, INV, Q / 2>(a);
    const T c1 = (T)0.98078528040323044912618223613424;   // cos(pi/16)
    const T s1 = (T)0.19509032201612826784828486847702;   // sin(pi/16)
    const T c3 = (T)0.83146961230254523707878837761791;   // cos(3 pi/16)
    const T s3 = (T)0.55557023301960222474283081394853;   // sin(3 pi/16)
    T c, s;   // w = c - i s (forward)
    if (Q == 1) { c = c1; s = s1; }
    else if (Q == 3) { c = c3; s = s3; }
    else if (Q == 5) { c = s3; s = c3; }
    else if (Q == 7) { c = s1; s = c1; }
    else if (Q == 9) { c = -s1; s = c1; }
    else if (Q == 11) { c = -s3; s = c3; }
    else if (Q == 13) { c = -c3; s = s3; }
    else { c = -c1; s = s1; }   // 15
    return cmul_cs<INV>(a, c, s);
}

// a[t] *= exp(-+ 2 pi i t/32), t = 0..15: the part of the half-sample shift w_P^(j + M t) of the odd
// half of a padded transform that depends on the register index (the w_P^j part rides in the
// stage twiddles, see load_twiddles_h).
template <typename T, bool INV> __device__ __forceinline__ void shift32(typename VT<T>::V *a)
{
    a[1] = mul_w32<T, INV, 1>(a[1]);
    a[2] = mul_w32<T, INV, 2>(a[2]);
    a[3] = mul_w32<T, INV, 3>(a[3]);
    a[4] = mul_w32<T, INV, 4>(a[4]);
    a[5] = mul_w32<T, INV, 5>(a[5]);
    a[6] = mul_w32<T, INV, 6>(a[6]);
    a[7] = mul_w32<T, INV, 7>(a[7]);
    a[8] = mul_w32<T, INV, 8>(a[8]);
    a[9] = mul_w32<T, INV, 9>(a[9]);
    a[10] = mul_w32<T, INV, 10>(a[10]);
    a[11] = mul_w32<T, INV, 11>(a[11]);
    a[12] = mul_w32<T, INV, 12>(a[12]);
    a[13] = mul_w32<T, INV, 13>(a[13]);
    a[14] = mul_w32<T, INV, 14>(a[14]);
    a[15] = mul_w32<T, INV, 15>(a[15]);
}

// Position <-> frequency of the in-register butterflies (DIF leaves digit-reversed order).
__host__ __device__ constexpr int rev16(int p) { return 4 * (p & 3) + (p >> 2); }
__host__ __device__ constexpr int rev8(int p) { return 4 * (p & 1) + (p >> 1); }
__host__ __device__ constexpr int revM(int M, int p)
{
    return M == 16 ? rev16(p) : M == 8 ? rev8(p) : p;   // dft4 / dft2 / identity are natural
}

// 16-point DFT.  Forward: natural in, position p holds frequency rev16(p).  Inverse (INV): the
// exact reverse (input in that order, natural out, unscaled).
template <typename T, bool INV> __device__ __forceinline__ void dft16(typename VT<T>::V *a)
{
    if (!INV) {
#pragma unroll
        for (int n1 = 0; n1 < 4; ++n1) dft4<false>(a[n1], a[n1 + 4], a[n1 + 8], a[n1 + 12]);
        a[5] = mul_w16<T, false, 1>(a[5]);
        a[9] = mul_w16<T, false, 2>(a[9]);
        a[13] = mul_w16<T, false, 3>(a[13]);
        a[6] = mul_w16<T, false, 2>(a[6]);
        a[10] = mul_w16<T, false, 4>(a[10]);
        a[14] = mul_w16<T, false, 6>(a[14]);
        a[7] = mul_w16<T, false, 3>(a[7]);
        a[11] = mul_w16<T, false, 6>(a[11]);
        a[15] = mul_w16<T, false, 9>(a[15]);
#pragma unroll
        for (int k2 = 0; k2 < 4; ++k2) dft4<false>(a[4 * k2], a[4 * k2 + 1], a[4 * k2 + 2], a[4 * k2 + 3]);
    } else {
#pragma unroll
        for (int k2 = 0; k2 < 4; ++k2) dft4<true>(a[4 * k2], a[4 * k2 + 1], a[4 * k2 + 2], a[4 * k2 + 3]);
        a[5] = mul_w16<T, true, 1>(a[5]);
        a[9] = mul_w16<T, true, 2>(a[9]);
        a[13] = mul_w16<T, true, 3>(a[13]);
        a[6] = mul_w16<T, true, 2>(a[6]);
        a[10] = mul_w16<T, true, 4>(a[10]);
        a[14] = mul_w16<T, true, 6>(a[14]);
        a[7] = mul_w16<T, true, 3>(a[7]);
        a[11] = mul_w16<T, true, 6>(a[11]);
        a[15] = mul_w16<T, true, 9>(a[15]);
#pragma unroll
        for (int n1 = 0; n1 < 4; ++n1) dft4<true>(a[n1], a[n1 + 4], a[n1 + 8], a[n1 + 12]);
    }
}

// 8-point DFT on a[0..7] with stride 1: forward natural in, position p holds rev8(p).
template <typename T, bool INV> __device__ __forceinline__ void dft8(typename VT<T>::V *a)
{
    if (!INV) {
        dft4<false>(a[0], a[2], a[4], a[6]);
        dft4<false>(a[1], a[3], a[5], a[7]);
        a[3] = mul_w16<T, false, 2>(a[3]);
        a[5] = mul_w16<T, false, 4>(a[5]);
        a[7] = mul_w16<T, false, 6>(a[7]);
        dft2(a[0], a[1]);
        dft2(a[2], a[3]);
        dft2(a[4], a[5]);
        dft2(a[6], a[7]);
    } else {
        dft2(a[0], a[1]);
        dft2(a[2], a[3]);
        dft2(a[4], a[5]);
        dft2(a[6], a[7]);
        a[3] = mul_w16<T, true, 2>(a[3]);
        a[5] = mul_w16<T, true, 4>(a[5]);
        a[7] = mul_w16<T, true, 6>(a[7]);
        dft4<true>(a[0], a[2], a[4], a[6]);
        dft4<true>(a[1], a[3], a[5], a[7]);
    }
}

// Stage 2: 16/M butterflies of radix M on slots [u*M, u*M + M).
template <typename T, bool INV, int M> __device__ __forceinline__ void dftM(typename VT<T>::V *a)
{
    if (M == 16) dft16<T, INV>(a);
    else if (M == 8) { dft8<T, INV>(a); dft8<T, INV>(a + 8); }
    else if (M == 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) dft4<INV>(a[4 * u], a[4 * u + 1], a[4 * u + 2], a[4 * u + 3]);
    } else if (M == 2) {
#pragma unroll
        for (int u = 0; u < 8; ++u) dft2(a[2 * u], a[2 * u + 1]);
    }
}

// Team geometry for N = 16 M.  Thread i of the team (0..15): stage 1 works on line l1 = i / M with
// elements j + M t (j = i % M); stage 2 on line l1 again with sub-transforms t' = q U + u (q = i % M).
template <int M> struct Team {
    static constexpr int N = 16 * M;
    static constexpr int U = 16 / M;        // radix-M butterflies per thread in stage 2
    static constexpr int LINES = 16 / M;    // lines per team
    // Complex elements of exchange scratch per team: 256 + 15 of skew, rounded so that the two
    // teams of a warp (lanes 2i and 2i+1 sit in the same half-warp) start 64 bytes apart modulo
    // the 128-byte bank period -- their simultaneous 64-bit (fp32) or 128-bit (fp64) accesses then
    // use disjoint halves of the banks.
    static constexpr int SCRATCH = 280;        // fp32: 280 * 8 B = 17.5 * 128 B
    static constexpr int SCRATCH64 = 276;      // fp64: 276 * 16 B = 34.5 * 128 B
};
template <typename T, int M> __host__ __device__ constexpr int team_scratch()
{
    return sizeof(T) == 8 ? Team<M>::SCRATCH64 : Team<M>::SCRATCH;
}

// frequency (0..N-1) of the N-point transform held in slot s = u*M + p of team thread with q = i % M
template <int M> __device__ __forceinline__ int slot_freq(int q, int s)
{
    const int u = s / M, p = s % M;
    return q * (16 / M) + u + 16 * revM(M, p);
}

__device__ __forceinline__ int skew(int lin) { return lin + (lin >> 4); }

// Twiddles of one team thread: tw[t'] = w_N^(j t') = w_P^(2 j t'), t' = 1..15 (tw[0] unused), from
// the table wP[q] = exp(-2 pi i q / P), P = 2N = 32 M.
template <typename T, int M>
__device__ __forceinline__ void load_twiddles2(typename VT<T>::V *tw, const typename VT<T>::V *__restrict__ wP, int j)
{
#pragma unroll
    for (int t = 1; t < 16; ++t) tw[t] = wP[(2 * j * t) & (32 * M - 1)];
}

// Twiddles of team half h with the half-sample shift of the odd half folded in:
// tw[t'] = w_N^(j t') w_P^(j h) = w_P^(j (2 t' + h)), t' = 0..15 (tw[0] = 1 for h = 0).  Used with
// fft_fwd/fft_inv<..., TW0 = true> and shift32 on the register index.
template <typename T, int M>
__device__ __forceinline__ void load_twiddles_h(typename VT<T>::V *tw, const typename VT<T>::V *__restrict__ wP, int j,
                                                int h)
{
#pragma unroll
    for (int t = 0; t < 16; ++t) tw[t] = wP[(j * (2 * t + h)) & (32 * M - 1)];
}

// Forward N-point transform of the team's lines.  a[t] = x[j + M t] on entry (natural), on exit
// slot s holds frequency slot_freq<M>(q, s).  `scr` = this team's scratch, i = team thread index.
template <typename T, int M, bool TW0 = false>
__device__ __forceinline__ void fft_fwd(typename VT<T>::V *a, const typename VT<T>::V *tw,
                                        typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    dft16<T, false>(a);
    if (M == 1) {
        // positions hold rev16 order; bring to slot order u = t' (U = 16)
        V b[16];
#pragma unroll
        for (int p = 0; p < 16; ++p) b[rev16(p)] = a[p];
#pragma unroll
        for (int p = 0; p < 16; ++p) a[p] = b[p];
        return;
    }
    const int l = i / M, j = i % M;
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        V v = a[p];
        if (tp != 0 || TW0) v = cmul(v, tw[tp]);
        scr[skew((l * 16 + tp) * M + j)] = v;
    }
    __syncwarp();
    constexpr int U = 16 / M;
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int u = s / M, jj = s % M;
        a[s] = scr[skew((l * 16 + j * U + u) * M + jj)];
    }
    dftM<T, false, M>(a);
}

// Inverse: slot order in, a[t] = N * x[j + M t] out (unscaled).
template <typename T, int M, bool TW0 = false>
__device__ __forceinline__ void fft_inv(typename VT<T>::V *a, const typename VT<T>::V *tw,
                                        typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    if (M == 1) {
        V b[16];
#pragma unroll
        for (int p = 0; p < 16; ++p) b[p] = a[rev16(p)];
#pragma unroll
        for (int p = 0; p < 16; ++p) a[p] = b[p];
        dft16<T, true>(a);
        return;
    }
    dftM<T, true, M>(a);
    const int l = i / M, j = i % M;
    constexpr int U = 16 / M;
    __syncwarp();
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int u = s / M, jj = s % M;
        scr[skew((l * 16 + j * U + u) * M + jj)] = a[s];
    }
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        V v = scr[skew((l * 16 + tp) * M + j)];
        if (tp != 0 || TW0) v = cmulc(v, tw[tp]);
        a[p] = v;
    }
    dft16<T, true>(a);
}

// The same transforms cut at the exchange, so that a caller holding several independent lines per
// thread (the three components of the z pass) can place the butterflies of one line between the
// scratch stores and loads of another:
//   forward  dft16 -> fwd_put | fwd_get -> dftM          inverse  dftM -> inv_put | inv_get -> dft16
template <typename T, int M, bool TW0>
__device__ __forceinline__ void fwd_put(const typename VT<T>::V *a, const typename VT<T>::V *tw,
                                        typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    const int l = i / M, j = i % M;
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        V v = a[p];
        if (tp != 0 || TW0) v = cmul(v, tw[tp]);
        scr[skew((l * 16 + tp) * M + j)] = v;
    }
}
template <typename T, int M>
__device__ __forceinline__ void fwd_get(typename VT<T>::V *a, const typename VT<T>::V *scr, int i)
{
    const int l = i / M, j = i % M;
    constexpr int U = 16 / M;
    __syncwarp();
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int u = s / M, jj = s % M;
        a[s] = scr[skew((l * 16 + j * U + u) * M + jj)];
    }
}
template <typename T, int M>
__device__ __forceinline__ void inv_put(const typename VT<T>::V *a, typename VT<T>::V *scr, int i)
{
    const int l = i / M, j = i % M;
    constexpr int U = 16 / M;
    __syncwarp();
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const int u = s / M, jj = s % M;
        scr[skew((l * 16 + j * U + u) * M + jj)] = a[s];
    }
}
template <typename T, int M, bool TW0>
__device__ __forceinline__ void inv_get(typename VT<T>::V *a, const typename VT<T>::V *tw,
                                        const typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    const int l = i / M, j = i % M;
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        V v = scr[skew((l * 16 + tp) * M + j)];
        if (tp != 0 || TW0) v = cmulc(v, tw[tp]);
        a[p] = v;
    }
}

// fwd_put / inv_get with the stage twiddles read from a shared-memory table instead of registers
// (fp64: 16 complex twiddles are 64 registers a thread holding three lines does not have):
// tws[t' * TWS] = the caller's twiddle t' of this lane (TW0 form, see load_twiddles_h).
template <typename T, int M, int TWS>
__device__ __forceinline__ void fwd_put_s(const typename VT<T>::V *a, const typename VT<T>::V *tws,
                                          typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    const int l = i / M, j = i % M;
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        scr[skew((l * 16 + tp) * M + j)] = cmul(a[p], tws[tp * TWS]);
    }
}
template <typename T, int M, int TWS>
__device__ __forceinline__ void inv_get_s(typename VT<T>::V *a, const typename VT<T>::V *tws,
                                          const typename VT<T>::V *scr, int i)
{
    typedef typename VT<T>::V V;
    const int l = i / M, j = i % M;
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        const int tp = rev16(p);
        a[p] = cmulc(scr[skew((l * 16 + tp) * M + j)], tws[tp * TWS]);
    }
}

// ---- lengths by template parameter M ------------------------------------------------------------------------
// M in {1, 2, 4, 8, 16}: N = 16 M, one team = 16 / M lines.  M = 12: N = 192 = 3 x 64, a radix-3 step on top of the
// M = 4 core: the line is split into its three decimated sub-sequences x_r[n'] = x[3 n' + r], which are three of the
// four lines of an M = 4 team (team thread i = 4 l + j: l = r, l = 3 idles); with G_r the padded 128-point transform
// of x_r,
//     X[k' + 128 s] = sum_r w_3^(r s) (w_384^(r k') G_r[k']),   k' < 128, s = 0, 1, 2,
// and the thread of sub-sequence l ends up with the outputs s = l of its slots (three lane exchanges per slot).
// The cropped inverse runs the same steps backwards.  wP is the table exp(-2 pi i q / P), P = 2 N, throughout.
template <int M> struct Len {
    static constexpr int N = 16 * M, P = 2 * N, MI = M, LT = 16 / M;
    static constexpr bool R3 = false;
};
template <> struct Len<12> {
    static constexpr int N = 192, P = 384, MI = 4, LT = 1;
    static constexpr bool R3 = true;
};

// element held in register t of team thread (l, j) on the data side
template <int M> __device__ __forceinline__ int len_elem(int l, int j, int t)
{
    return Len<M>::R3 ? 3 * (j + Len<M>::MI * t) + l : j + M * t;
}
// index into wP of the odd half's pre-twiddle of that element: w_P'^(n') of the transform the core runs
template <int M> __device__ __forceinline__ int len_pre(int l, int j, int t)
{
    return Len<M>::R3 ? 3 * (j + Len<M>::MI * t) : j + M * t;
}
// frequency (0..P-1) held in slot s of team thread (l, j), half h, on the spectral side
template <int M> __device__ __forceinline__ int len_freq(int l, int j, int s, int h)
{
    return 2 * slot_freq<Len<M>::MI>(j, s) + h + (Len<M>::R3 ? 128 * l : 0);
}
template <typename T, int M>
__device__ __forceinline__ void len_twiddles(typename VT<T>::V *tw, const typename VT<T>::V *__restrict__ wP, int j)
{
    if (Len<M>::R3) {
#pragma unroll
        for (int t = 1; t < 16; ++t) tw[t] = wP[(6 * j * t) % 384];         // w_64^(j t)
    } else {
        load_twiddles2<T, Len<M>::MI>(tw, wP, j);
    }
}

// the value slot holds in the thread of sub-sequence r of the same (j, h): lane = 8 l + 2 j + h
template <typename V> __device__ __forceinline__ V shfl_sub(V v, int lane, int r)
{
    V o;
    o.x = __shfl_sync(0xffffffffu, v.x, (lane & 7) + 8 * r);
    o.y = __shfl_sync(0xffffffffu, v.y, (lane & 7) + 8 * r);
    return o;
}

// X_l = T_0 + w^l T_1 + w^(2l) T_2 with w = exp(-+ 2 pi i / 3) (forward / INV), for the thread's own l
template <typename T, bool INV, typename V> __device__ __forceinline__ V dft3_own(V t0, V t1, V t2, int l)
{
    const V sm = cadd(t1, t2), df = csub(t1, t2);
    const T hs = (T)0.86602540378443864676372317075294;
    // l = 0: t0 + sm;  l = 1, 2: t0 - sm / 2 -+ i hs df (forward: l = 1 takes -i), inverse the other way round
    const T cs = l == 0 ? (T)1 : (T)-0.5;
    T g = l == 0 ? (T)0 : (l == 1 ? -hs : hs);
    if (INV) g = -g;
    // (re, im) = t0 + cs sm + g (-df.y, df.x): two packed multiply-adds
    return pfma(mk<T>(df.y, df.x), mk<T>(-g, g), pfma(sm, mk<T>(cs, cs), t0));
}

template <typename T, int M>
__device__ __forceinline__ void len_fwd(typename VT<T>::V *a, const typename VT<T>::V *tw, typename VT<T>::V *scr, int i,
                                        const typename VT<T>::V *__restrict__ wP, int lane)
{
    typedef typename VT<T>::V V;
    fft_fwd<T, Len<M>::MI>(a, tw, scr, i);
    if (Len<M>::R3) {
        const int l = min(i >> 2, 2), j = i & 3, h = lane & 1;
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int kp = 2 * slot_freq<4>(j, s) + h;
            const V v = cmul(a[s], wP[l * kp]);
            a[s] = dft3_own<T, false>(shfl_sub(v, lane, 0), shfl_sub(v, lane, 1), shfl_sub(v, lane, 2), l);
        }
    }
}

template <typename T, int M>
__device__ __forceinline__ void len_inv(typename VT<T>::V *a, const typename VT<T>::V *tw, typename VT<T>::V *scr, int i,
                                        const typename VT<T>::V *__restrict__ wP, int lane)
{
    typedef typename VT<T>::V V;
    if (Len<M>::R3) {
        const int l = min(i >> 2, 2), j = i & 3, h = lane & 1;
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            const int kp = 2 * slot_freq<4>(j, s) + h;
            const V y = dft3_own<T, true>(shfl_sub(a[s], lane, 0), shfl_sub(a[s], lane, 1), shfl_sub(a[s], lane, 2), l);
            a[s] = cmulc(y, wP[l * kp]);
        }
    }
    fft_inv<T, Len<M>::MI>(a, tw, scr, i);
}

// The radix-3 step of Len<12> with two lane exchanges per slot (the pipelined 192-cell kernels): a thread keeps its
// own value and fetches those of the sub-sequences l + 1 and l + 2 (mod 3); `lane` = 8 l + 2 j + h, l = min(i / 4, 2).
template <typename T, bool INV>
__device__ __forceinline__ typename VT<T>::V r3_gather(typename VT<T>::V own, int lane, int l)
{
    typedef typename VT<T>::V V;
    const int la = (lane & 7) + 8 * (l == 2 ? 0 : l + 1), lb = (lane & 7) + 8 * (l == 0 ? 2 : l - 1);
    V A, B;                                                     // values of sub-sequences l + 1 and l + 2
    A.x = __shfl_sync(0xffffffffu, own.x, la);
    A.y = __shfl_sync(0xffffffffu, own.y, la);
    B.x = __shfl_sync(0xffffffffu, own.x, lb);
    B.y = __shfl_sync(0xffffffffu, own.y, lb);
    // (t0, t1, t2) = l = 0: (own, A, B); l = 1: (B, own, A); l = 2: (A, B, own) -- scalar selects, no branches
    const bool p0 = l == 0, p1 = l == 1;
    const V t0 = mk<T>(p0 ? own.x : (p1 ? B.x : A.x), p0 ? own.y : (p1 ? B.y : A.y));
    const V t1 = mk<T>(p0 ? A.x : (p1 ? own.x : B.x), p0 ? A.y : (p1 ? own.y : B.y));
    const V t2 = mk<T>(p0 ? B.x : (p1 ? A.x : own.x), p0 ? B.y : (p1 ? A.y : own.y));
    return dft3_own<T, INV>(t0, t1, t2, l);
}
// The twiddle w_384^(l k') of slot s = 4 u + p, k' = 8 j + 2 u + 32 p + h, factors into w^(l (2 t' + h)), t' = 4 j + u
// the position the value had in the exchange -- which the caller folds into its stage twiddles,
// tw[t'] = w_384^((3 j + l)(2 t' + h)) -- and bc[p - 1] = w_12^(l p), applied here (12 products per transform).
template <typename T>
__device__ __forceinline__ void r3_fwd(typename VT<T>::V *a, const typename VT<T>::V *bc, int lane, int l)
{
#pragma unroll
    for (int s = 0; s < 16; ++s) a[s] = r3_gather<T, false>((s & 3) ? cmul(a[s], bc[(s & 3) - 1]) : a[s], lane, l);
}
template <typename T>
__device__ __forceinline__ void r3_inv(typename VT<T>::V *a, const typename VT<T>::V *bc, int lane, int l)
{
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const typename VT<T>::V y = r3_gather<T, true>(a[s], lane, l);
        a[s] = (s & 3) ? cmulc(y, bc[(s & 3) - 1]) : y;
    }
}

} // namespace nmf
