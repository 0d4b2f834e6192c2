// Shared-memory mixed-radix FFT stages (device code).
//
// a2/a4 of the hot path: the zero-padded transforms of the demag convolution
// (PAPER.md:175-181).  Forward = decimation in frequency, inverse = its adjoint stage by stage,
// so no reordering pass exists anywhere: spectra live in digit-reversed position order and the
// tensor multiply looks the frequency of a position up in a table (NmFftPlan, nm_internal.h).
// Every butterfly reads and writes the same shared-memory slots, so a stage is in place with one
// block barrier after it.
#pragma once

#include "nm_internal.h"

template <typename T> struct Cx {
    typedef typename NmVec2<T>::type V;
    static __device__ __forceinline__ V make(T a, T b)
    {
        V v;
        v.x = a;
        v.y = b;
        return v;
    }
    static __device__ __forceinline__ V add(V a, V b) { return make(a.x + b.x, a.y + b.y); }
    static __device__ __forceinline__ V sub(V a, V b) { return make(a.x - b.x, a.y - b.y); }
    static __device__ __forceinline__ V mul(V a, V b)
    {
        return make(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
    }
    static __device__ __forceinline__ V mulc(V a, V b)   // a * conj(b)
    {
        return make(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
    }
    // multiply by -i (forward) or +i (inverse)
    template <bool INV> static __device__ __forceinline__ V rot90(V a)
    {
        return INV ? make(-a.y, a.x) : make(a.y, -a.x);
    }
};

// R-point DFT in registers, sign -1 (INV = false) or +1 (INV = true), no scaling.
template <typename T, bool INV>
__device__ __forceinline__ void dft2(typename Cx<T>::V *x)
{
    typedef Cx<T> C;
    typename C::V a = x[0], b = x[1];
    x[0] = C::add(a, b);
    x[1] = C::sub(a, b);
}

template <typename T, bool INV>
__device__ __forceinline__ void dft3(typename Cx<T>::V *x)
{
    typedef Cx<T> C;
    const T h = (T)0.86602540378443864676372317075294;   // sin(pi/3)
    typename C::V s = C::add(x[1], x[2]);
    typename C::V d = C::sub(x[1], x[2]);
    typename C::V m = C::make(x[0].x - (T)0.5 * s.x, x[0].y - (T)0.5 * s.y);
    // forward: y1 = m - i h d, y2 = m + i h d ; inverse: swapped
    typename C::V r = C::make(h * d.y, -h * d.x);          // -i h d
    x[0] = C::add(x[0], s);
    if (!INV) {
        x[1] = C::add(m, r);
        x[2] = C::sub(m, r);
    } else {
        x[1] = C::sub(m, r);
        x[2] = C::add(m, r);
    }
}

template <typename T, bool INV>
__device__ __forceinline__ void dft4(typename Cx<T>::V *x)
{
    typedef Cx<T> C;
    typename C::V a = C::add(x[0], x[2]), b = C::sub(x[0], x[2]);
    typename C::V c = C::add(x[1], x[3]), d = C::template rot90<INV>(C::sub(x[1], x[3]));
    x[0] = C::add(a, c);
    x[2] = C::sub(a, c);
    x[1] = C::add(b, d);
    x[3] = C::sub(b, d);
}

template <typename T, bool INV>
__device__ __forceinline__ void dft8(typename Cx<T>::V *x)
{
    typedef Cx<T> C;
    typename C::V e[4] = {x[0], x[2], x[4], x[6]};
    typename C::V o[4] = {x[1], x[3], x[5], x[7]};
    dft4<T, INV>(e);
    dft4<T, INV>(o);
    const T q = (T)0.70710678118654752440084436210485;
    // o[k] *= w8^k, w8 = exp(-+ i pi/4)
    typename C::V t1 = INV ? C::make(q * (o[1].x - o[1].y), q * (o[1].x + o[1].y))
                           : C::make(q * (o[1].x + o[1].y), q * (o[1].y - o[1].x));
    typename C::V t2 = C::template rot90<INV>(o[2]);
    typename C::V t3 = INV ? C::make(-q * (o[3].x + o[3].y), q * (o[3].x - o[3].y))
                           : C::make(q * (o[3].y - o[3].x), -q * (o[3].x + o[3].y));
    x[0] = C::add(e[0], o[0]);
    x[4] = C::sub(e[0], o[0]);
    x[1] = C::add(e[1], t1);
    x[5] = C::sub(e[1], t1);
    x[2] = C::add(e[2], t2);
    x[6] = C::sub(e[2], t2);
    x[3] = C::add(e[3], t3);
    x[7] = C::sub(e[3], t3);
}

// Odd prime radix (5, 7): the R-point DFT by its definition, y_k = sum_t x_t w^(k t mod R) with
// w^q = exp(-/+ 2 pi i q / R) = tw[q L / R] (conjugated for the inverse) read from the table of
// the whole transform.
template <typename T, bool INV, int R>
__device__ __forceinline__ void dft_prime(typename Cx<T>::V *x, const typename Cx<T>::V *__restrict__ tw, int L)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    V w[R];
    const int step = L / R;
#pragma unroll
    for (int q = 1; q < R; ++q) w[q] = tw[q * step];
    V y[R];
    y[0] = x[0];
#pragma unroll
    for (int t = 1; t < R; ++t) y[0] = C::add(y[0], x[t]);
#pragma unroll
    for (int k = 1; k < R; ++k) {
        V acc = x[0];
#pragma unroll
        for (int t = 1; t < R; ++t)
            acc = C::add(acc, INV ? C::mulc(x[t], w[(k * t) % R]) : C::mul(x[t], w[(k * t) % R]));
        y[k] = acc;
    }
#pragma unroll
    for (int k = 0; k < R; ++k) x[k] = y[k];
}

template <typename T, bool INV, int R>
__device__ __forceinline__ void dftR(typename Cx<T>::V *x)
{
    if (R == 2) dft2<T, INV>(x);
    else if (R == 3) dft3<T, INV>(x);
    else if (R == 4) dft4<T, INV>(x);
    else dft8<T, INV>(x);
}

// One stage on `n_lines` lines held in shared memory.
//   element e of line l lives at s[l * line_stride + e * elem_stride]
//   n = current block length (forward: before the stage; inverse: after it), m = n / R
//   tw[q] = exp(-2 pi i q / L)
// LINE_FAST: consecutive threads take consecutive lines (strided y/z layouts), else consecutive
// butterflies of one line (x layout).
template <typename T, bool INV, int R, bool LINE_FAST>
__device__ __forceinline__ void fft_stage(typename Cx<T>::V *s, int n_lines, int line_stride,
                                          int elem_stride, int L, int n,
                                          const typename Cx<T>::V *__restrict__ tw)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    const int m = n / R;
    const int per_line = L / R;
    const int total = n_lines * per_line;
    const int tw_step = L / n;
    for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
        int line, bf;
        if (LINE_FAST) {
            line = idx % n_lines;
            bf = idx / n_lines;
        } else {
            bf = idx % per_line;
            line = idx / per_line;
        }
        const int blk = bf / m, j = bf - blk * m;
        V *p = s + line * line_stride + (blk * n + j) * elem_stride;
        const int es = m * elem_stride;
        V x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) x[t] = p[t * es];
        if (INV) {
#pragma unroll
            for (int t = 1; t < R; ++t) x[t] = C::mulc(x[t], tw[j * t * tw_step]);
        }
        if (R == 5 || R == 7) dft_prime<T, INV, R>(x, tw, L);
        else dftR<T, INV, R>(x);
        if (!INV) {
#pragma unroll
            for (int t = 1; t < R; ++t) x[t] = C::mul(x[t], tw[j * t * tw_step]);
        }
#pragma unroll
        for (int t = 0; t < R; ++t) p[t * es] = x[t];
    }
}

// PR: the transform may contain radix-5 / 7 stages (kernels for 2^a 3^b lengths are compiled without
// them, so their register allocation does not pay for the prime butterflies).
template <typename T, bool INV, bool LINE_FAST, bool PR>
__device__ __forceinline__ void fft_stage_any(int R, typename Cx<T>::V *s, int n_lines,
                                              int line_stride, int elem_stride, int L, int n,
                                              const typename Cx<T>::V *__restrict__ tw)
{
    switch (R) {
    case 2: fft_stage<T, INV, 2, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    case 3: fft_stage<T, INV, 3, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    case 4: fft_stage<T, INV, 4, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    case 5: if (PR) fft_stage<T, INV, 5, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    case 7: if (PR) fft_stage<T, INV, 7, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    default: fft_stage<T, INV, 8, LINE_FAST>(s, n_lines, line_stride, elem_stride, L, n, tw); break;
    }
}

// Whole transform of n_lines lines in shared memory.  Caller must __syncthreads() before (data
// visible) — a barrier follows every stage, so results are visible on return.
template <typename T, bool LINE_FAST, bool PR>
__device__ __forceinline__ void fft_forward(typename Cx<T>::V *s, int n_lines, int line_stride,
                                            int elem_stride, const NmFftPlan &plan,
                                            const typename Cx<T>::V *__restrict__ tw)
{
    int n = plan.L;
    for (int st = 0; st < plan.n_stages; ++st) {
        const int R = plan.radix[st];
        fft_stage_any<T, false, LINE_FAST, PR>(R, s, n_lines, line_stride, elem_stride, plan.L, n, tw);
        n /= R;
        __syncthreads();
    }
}

template <typename T, bool LINE_FAST, bool PR>
__device__ __forceinline__ void fft_inverse(typename Cx<T>::V *s, int n_lines, int line_stride,
                                            int elem_stride, const NmFftPlan &plan,
                                            const typename Cx<T>::V *__restrict__ tw)
{
    int n = 1;
    for (int st = plan.n_stages - 1; st >= 0; --st) {
        const int R = plan.radix[st];
        n *= R;
        fft_stage_any<T, true, LINE_FAST, PR>(R, s, n_lines, line_stride, elem_stride, plan.L, n, tw);
        __syncthreads();
    }
}
