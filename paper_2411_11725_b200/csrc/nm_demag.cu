// Demagnetisation field on cells: a1-a4 of the hot path.
//
// node->cell averaging, zero-padded FFT convolution with the demag tensor of
// uniformly magnetised cuboids, (cell->node averaging happens in nm_local.cu).  Reading C5:
//   M_c = Ms_c (1/8) sum_i m_{c+i},   H_c = - sum_c' N(c - c') M_c',   P_d = 2 N_d (1 if N_d = 1).
//
// Passes (spectra in digit-reversed position order along y and z, natural order along x):
//   k_x_fwd      nodes -> A[3][N3][N2][C1p]      average * Ms, real-to-complex along x through one
//                                                complex transform of length N1 = P1/2
//   k_lines_fwd  A -> B[3][N3][P2][C1p]          y transform (3-D meshes only)
//   k_mid        in place on B (z) or A (y)      forward, H^ = -N^ M^, inverse, in shared memory
//   k_lines_inv  B -> A                          inverse y, cropped to N2
//   k_x_inv      A -> Hc[3][N3][N2][N1]          complex-to-real along x, cropped to N1
// The factor 1/(P1 P2 P3) lives in N^.
#include "nm_fft.cuh"
#include "nm_internal.h"

namespace {

template <typename T> struct Tile {
    static constexpr int lines_y = sizeof(T) == 4 ? 16 : 8;   // k1 columns per CTA, y passes
    static constexpr int lines_mid = sizeof(T) == 4 ? 8 : 4;  // k1 columns per CTA, middle pass
};

constexpr int kThreads = 256;
constexpr int kRowsX = 4;   // cell rows (c2) per CTA in the x passes (2 where that leaves SMs without a CTA)

// ---------------------------------------------------------------------------------------------
template <typename T, int RX, bool PR>
__global__ void __launch_bounds__(kThreads)
k_x_fwd(const T *__restrict__ fld, const T *__restrict__ Ms, typename Cx<T>::V *__restrict__ A,
        NmGeom g, NmFftPlan plan, const typename Cx<T>::V *__restrict__ tw,
        const typename Cx<T>::V *__restrict__ tw2, const int *__restrict__ pos)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s = reinterpret_cast<V *>(smem_raw);
    const int Lx = g.Lx;
    const int c3 = blockIdx.y;
    const int row0 = blockIdx.x * RX;
    const int n_lines = 3 * RX;
    const long long plane = g.zs;      // 0 / g.ys = 0 along an axis the basis does not vary in (Eqs. 23-24):
    const int rowp = g.ys;             // the four (dy, dz) nodes of a cell column then coincide pairwise
    // 1. cell averages, packed two reals per complex slot
    for (int idx = threadIdx.x; idx < n_lines * Lx; idx += blockDim.x) {
        const int n = idx % Lx;
        const int line = idx / Lx;
        const int r = line % RX, comp = line / RX;
        const int c2 = row0 + r;
        T v0 = 0, v1 = 0;
        if (c2 < g.N2) {
            const T *base = fld + (long long)comp * g.nodes + (long long)c3 * plane +
                            (long long)c2 * rowp;
            const int c1 = 2 * n;
            if (c1 < g.N1) {
                // column sums over the 4 (dy,dz) nodes at x = c1, c1+1, c1+2
                T col[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const int x = c1 + d;
                    col[d] = x <= g.N1 ? (base[x] + base[x + rowp]) + (base[x + plane] + base[x + plane + rowp])
                                       : (T)0;
                }
                const long long cell = ((long long)c3 * g.N2 + c2) * g.N1 + c1;
                v0 = Ms[cell] * (T)0.125 * (col[0] + col[1]);
                if (c1 + 1 < g.N1) v1 = Ms[cell + 1] * (T)0.125 * (col[1] + col[2]);
            }
        }
        s[line * Lx + n] = C::make(v0, v1);
    }
    __syncthreads();
    // 2. complex transform of length Lx
    fft_forward<T, false, PR>(s, n_lines, Lx, 1, plan, tw);
    // 3. untangle: X[k] = 1/2 [(Z[k] + conj Z[Lx-k]) - i W^k (Z[k] - conj Z[Lx-k])], k = 0..N1
    for (int idx = threadIdx.x; idx < n_lines * g.C1; idx += blockDim.x) {
        const int k = idx % g.C1;
        const int line = idx / g.C1;
        const int r = line % RX, comp = line / RX;
        const int c2 = row0 + r;
        if (c2 >= g.N2) continue;
        const V *ln = s + line * Lx;
        const V zk = ln[pos[k == Lx ? 0 : k]];
        const V zm = ln[pos[k == 0 ? 0 : Lx - k]];
        const V e = C::make(zk.x + zm.x, zk.y - zm.y);      // Z[k] + conj Z[-k]
        const V o = C::make(zk.x - zm.x, zk.y + zm.y);      // Z[k] - conj Z[-k]
        const V wo = C::mul(tw2[k], o);
        // -i * wo = (wo.y, -wo.x)
        const V X = C::make((T)0.5 * (e.x + wo.y), (T)0.5 * (e.y - wo.x));
        A[(((long long)comp * g.N3 + c3) * g.N2 + c2) * g.C1p + k] = X;
    }
}

template <typename T, int RX, bool PR>
__global__ void __launch_bounds__(kThreads)
k_x_inv(const typename Cx<T>::V *__restrict__ A, T *__restrict__ Hc, NmGeom g, NmFftPlan plan,
        const typename Cx<T>::V *__restrict__ tw, const typename Cx<T>::V *__restrict__ tw2,
        const int *__restrict__ pos)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s = reinterpret_cast<V *>(smem_raw);
    const int Lx = g.Lx;
    const int c3 = blockIdx.y;
    const int row0 = blockIdx.x * RX;
    const int n_lines = 3 * RX;
    // 1. Z'[k] = (X[k] + conj X[Lx-k]) + i conj(W^k) (X[k] - conj X[Lx-k]), stored at its position
    for (int idx = threadIdx.x; idx < n_lines * Lx; idx += blockDim.x) {
        const int k = idx % Lx;
        const int line = idx / Lx;
        const int r = line % RX, comp = line / RX;
        const int c2 = row0 + r;
        V z = C::make((T)0, (T)0);
        if (c2 < g.N2) {
            const V *row = A + (((long long)comp * g.N3 + c3) * g.N2 + c2) * g.C1p;
            if (g.N1 == 1) {
                z = C::make(row[0].x, (T)0);
            } else {
                const V xk = row[k];
                const V xm = row[Lx - k];
                const V e = C::make(xk.x + xm.x, xk.y - xm.y);
                const V o = C::make(xk.x - xm.x, xk.y + xm.y);
                const V wo = C::mulc(o, tw2[k]);             // conj(W^k) * o
                z = C::make(e.x - wo.y, e.y + wo.x);         // e + i wo
            }
        }
        s[line * Lx + pos[k]] = z;
    }
    __syncthreads();
    fft_inverse<T, false, PR>(s, n_lines, Lx, 1, plan, tw);
    // 2. x[2n] = Re z[n], x[2n+1] = Im z[n], cropped to N1
    for (int idx = threadIdx.x; idx < n_lines * g.N1; idx += blockDim.x) {
        const int c1 = idx % g.N1;
        const int line = idx / g.N1;
        const int r = line % RX, comp = line / RX;
        const int c2 = row0 + r;
        if (c2 >= g.N2) continue;
        const V z = s[line * Lx + (c1 >> 1)];
        Hc[(long long)comp * g.cells + ((long long)c3 * g.N2 + c2) * g.N1 + c1] = (c1 & 1) ? z.y : z.x;
    }
}

// ---------------------------------------------------------------------------------------------
// y transform of one (component, c3) slab for a tile of k1 columns.
template <typename T, bool INV, bool PR>
__global__ void __launch_bounds__(kThreads)
k_lines(const typename Cx<T>::V *__restrict__ src, typename Cx<T>::V *__restrict__ dst, NmGeom g,
        int bt, NmFftPlan plan, const typename Cx<T>::V *__restrict__ tw)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s = reinterpret_cast<V *>(smem_raw);
    const int k0 = blockIdx.x * bt;
    const int c3 = blockIdx.y, comp = blockIdx.z;
    const int P = g.P2, N = g.N2;
    const long long slabA = ((long long)comp * g.N3 + c3) * N * g.C1p;
    const long long slabB = ((long long)comp * g.N3 + c3) * P * g.C1p;
    const int n_in = INV ? P : N;
    for (int idx = threadIdx.x; idx < P * bt; idx += blockDim.x) {
        const int b = idx % bt, e = idx / bt;
        V v = C::make((T)0, (T)0);
        if (e < n_in && k0 + b < g.C1p) v = src[(INV ? slabB : slabA) + (long long)e * g.C1p + k0 + b];
        s[idx] = v;
    }
    __syncthreads();
    if (INV) fft_inverse<T, true, PR>(s, bt, 1, bt, plan, tw);
    else fft_forward<T, true, PR>(s, bt, 1, bt, plan, tw);
    const int n_out = INV ? N : P;
    for (int idx = threadIdx.x; idx < n_out * bt; idx += blockDim.x) {
        const int b = idx % bt, e = idx / bt;
        if (k0 + b < g.C1p) dst[(INV ? slabA : slabB) + (long long)e * g.C1p + k0 + b] = s[idx];
    }
}

// ---------------------------------------------------------------------------------------------
// Middle pass: for a tile of k1 columns and one fixed index of the other axis, transform the
// three components along the last untransformed axis, apply H^ = -N^ M^ and transform back.
struct MidArgs {
    long long comp_stride;    // complex elements between components
    long long elem_stride;    // complex elements between consecutive line elements
    long long fixed_stride;   // complex elements per step of blockIdx.y's index
    int N, P;                 // loaded / padded length
    int axis;                 // 2: line along z (3-D), 1: line along y (single-layer)
    int n_fixed;              // extent of the fixed index (P2 in 3-D, 1 otherwise)
};

template <typename T, bool PR>
__global__ void __launch_bounds__(kThreads)
k_mid(typename Cx<T>::V *__restrict__ buf, const T *__restrict__ Nhat, NmGeom g, MidArgs a, int bt,
      NmFftPlan plan, const typename Cx<T>::V *__restrict__ tw, const int *__restrict__ kmap_line,
      const int *__restrict__ kmap_fixed, const int *__restrict__ pos_fixed)
{
    typedef Cx<T> C;
    typedef typename C::V V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V *s = reinterpret_cast<V *>(smem_raw);
    const int k0 = blockIdx.x * bt;
    const int n_lines = 3 * bt;
    // fixed index: frequencies +k and -k of the other axis in neighbouring CTAs (they read the
    // same folded tensor rows, so the second read hits L2)
    int kf = 0, pf = 0;
    if (a.n_fixed > 1) {
        const int j = blockIdx.y;
        kf = (j & 1) ? a.n_fixed - ((j + 1) >> 1) : (j >> 1);
        pf = pos_fixed[kf];
    }
    V *base = buf + (long long)pf * a.fixed_stride + k0;
    for (int idx = threadIdx.x; idx < a.P * n_lines; idx += blockDim.x) {
        const int l = idx % n_lines, e = idx / n_lines;
        const int b = l % bt, comp = l / bt;
        V v = C::make((T)0, (T)0);
        if (e < a.N && k0 + b < g.C1p) v = base[comp * a.comp_stride + e * a.elem_stride + b];
        s[idx] = v;
    }
    __syncthreads();
    fft_forward<T, true, PR>(s, n_lines, 1, n_lines, plan, tw);
    // tensor multiply
    const long long tcomp = (long long)g.K3 * g.K2 * g.C1p;
    int kk_fixed = 0;
    T s_fixed = (T)1;
    if (a.n_fixed > 1) {
        const int half = a.n_fixed >> 1;
        kk_fixed = kf > half ? a.n_fixed - kf : kf;
        if (kf > half) s_fixed = (T)-1;
    }
    for (int idx = threadIdx.x; idx < a.P * bt; idx += blockDim.x) {
        const int b = idx % bt, e = idx / bt;
        if (k0 + b >= g.C1p) continue;
        const int kl = kmap_line[e];
        const int half = a.P >> 1;
        const int kk_line = kl > half ? a.P - kl : kl;
        const T s_line = kl > half ? (T)-1 : (T)1;
        int kk2, kk3;
        T sy, sz;
        if (a.axis == 2) {
            kk3 = kk_line; sz = s_line; kk2 = kk_fixed; sy = s_fixed;
        } else {
            kk2 = kk_line; sy = s_line; kk3 = 0; sz = (T)1;
        }
        const T *tn = Nhat + ((long long)kk3 * g.K2 + kk2) * g.C1p + k0 + b;
        const T nxx = tn[0], nyy = tn[tcomp], nzz = tn[2 * tcomp];
        const T nxy = sy * tn[3 * tcomp], nxz = sz * tn[4 * tcomp], nyz = sy * sz * tn[5 * tcomp];
        V *p = s + e * n_lines + b;
        const V mx = p[0], my = p[bt], mz = p[2 * bt];
        p[0] = C::make(-(nxx * mx.x + nxy * my.x + nxz * mz.x), -(nxx * mx.y + nxy * my.y + nxz * mz.y));
        p[bt] = C::make(-(nxy * mx.x + nyy * my.x + nyz * mz.x), -(nxy * mx.y + nyy * my.y + nyz * mz.y));
        p[2 * bt] = C::make(-(nxz * mx.x + nyz * my.x + nzz * mz.x), -(nxz * mx.y + nyz * my.y + nzz * mz.y));
    }
    __syncthreads();
    fft_inverse<T, true, PR>(s, n_lines, 1, n_lines, plan, tw);
    for (int idx = threadIdx.x; idx < a.N * n_lines; idx += blockDim.x) {
        const int l = idx % n_lines, e = idx / n_lines;
        const int b = l % bt, comp = l / bt;
        if (k0 + b < g.C1p) base[comp * a.comp_stride + e * a.elem_stride + b] = s[idx];
    }
}

template <typename K> nm_status set_smem(K kernel, size_t bytes)
{
    if (bytes > 48 * 1024)
        NM_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return NM_OK;
}

} // namespace

// Largest shared-memory footprint allowed per CTA for these passes
static const size_t kSmemCap = 200 * 1024;

static bool has_prime_radix(const NmFftPlan &p)
{
    for (int s = 0; s < p.n_stages; ++s)
        if (p.radix[s] == 5 || p.radix[s] == 7) return true;
    return false;
}

template <typename T, bool PR> nm_status conv_general(nm_mesh *mesh, const T *fld, T *Hc_out, cudaStream_t st);

template <typename T>
nm_status nm_demag_conv(nm_mesh *mesh, const T *fld, T *Hc_out, cudaStream_t st)
{
    if (mesh->fast.on) return nm_demag_conv_fast<T>(mesh, fld, Hc_out, st);
    // lengths 2^a 3^b keep the kernels without the radix-5 / 7 butterflies
    const bool pr = has_prime_radix(mesh->plan_x) || has_prime_radix(mesh->plan_y) || has_prime_radix(mesh->plan_z);
    return pr ? conv_general<T, true>(mesh, fld, Hc_out, st) : conv_general<T, false>(mesh, fld, Hc_out, st);
}

template <typename T, bool PR>
nm_status conv_general(nm_mesh *mesh, const T *fld, T *Hc_out, cudaStream_t st)
{
    typedef typename Cx<T>::V V;
    const NmGeom &g = mesh->g;
    V *A = (V *)mesh->bufA, *B = (V *)mesh->bufB;
    // x passes: 4 cell rows per CTA, or 2 where 4 would leave fewer than two CTAs per SM (films)
    const bool rx2 = (long long)((g.N2 + kRowsX - 1) / kRowsX) * g.N3 < 2LL * mesh->sm_count;
    const int RXv = rx2 ? 2 : kRowsX;
    const dim3 gx((g.N2 + RXv - 1) / RXv, g.N3);
    const size_t smx = (size_t)3 * RXv * g.Lx * sizeof(V);
    if (smx > kSmemCap) {
        nm_set_error("N1 = %d too long for the x pass", g.N1);
        return NM_EUNSUPPORTED;
    }
    {
        NmLaunchScope sc(mesh, NM_K_X_FWD, st);
        if (rx2) {
            NM_TRY(set_smem(k_x_fwd<T, 2, PR>, smx));
            k_x_fwd<T, 2, PR><<<gx, kThreads, smx, st>>>(fld, (const T *)mesh->Ms, A, g, mesh->plan_x,
                                                    (const V *)mesh->tw_x, (const V *)mesh->tw_x2, mesh->pos_x);
        } else {
            NM_TRY(set_smem(k_x_fwd<T, kRowsX, PR>, smx));
            k_x_fwd<T, kRowsX, PR><<<gx, kThreads, smx, st>>>(fld, (const T *)mesh->Ms, A, g, mesh->plan_x,
                                                         (const V *)mesh->tw_x, (const V *)mesh->tw_x2, mesh->pos_x);
        }
    }


    MidArgs ma;
    V *midbuf;
    const NmFftPlan *mplan;
    const V *mtw;
    const int *kline;
    if (g.N3 > 1) {
        int bt = Tile<T>::lines_y;
        while ((size_t)g.P2 * bt * sizeof(V) > kSmemCap && bt > 1) bt >>= 1;
        const size_t smy = (size_t)g.P2 * bt * sizeof(V);
        if (smy > kSmemCap) {
            nm_set_error("N2 = %d too long for the y pass", g.N2);
            return NM_EUNSUPPORTED;
        }
        NM_TRY(set_smem(k_lines<T, false, PR>, smy));
        NM_TRY(set_smem(k_lines<T, true, PR>, smy));
        const dim3 gy((g.C1p + bt - 1) / bt, g.N3, 3);
        {
            NmLaunchScope sc(mesh, NM_K_Y_FWD, st);
            k_lines<T, false, PR><<<gy, kThreads, smy, st>>>(A, B, g, bt, mesh->plan_y, (const V *)mesh->tw_y);
        }

        ma.comp_stride = (long long)g.N3 * g.P2 * g.C1p;
        ma.elem_stride = (long long)g.P2 * g.C1p;
        ma.fixed_stride = g.C1p;
        ma.N = g.N3; ma.P = g.P3; ma.axis = 2; ma.n_fixed = g.P2;
        midbuf = B; mplan = &mesh->plan_z; mtw = (const V *)mesh->tw_z; kline = mesh->kmap_z;
    } else {
        ma.comp_stride = (long long)g.N2 * g.C1p;
        ma.elem_stride = g.C1p;
        ma.fixed_stride = 0;
        ma.N = g.N2; ma.P = g.P2; ma.axis = 1; ma.n_fixed = 1;
        midbuf = A; mplan = &mesh->plan_y; mtw = (const V *)mesh->tw_y; kline = mesh->kmap_y;
    }
    {
        int bt = Tile<T>::lines_mid;
        while ((size_t)3 * ma.P * bt * sizeof(V) > kSmemCap && bt > 1) bt >>= 1;
        // single-layer films have C1p / bt CTAs only: narrower tiles (down to two columns) until
        // there are two CTAs per SM (512 x 512 x 1: 0.105 -> 0.048 ms)
        if (ma.n_fixed == 1)
            while (bt > 2 && (g.C1p + bt - 1) / bt < 2 * mesh->sm_count) bt >>= 1;
        const size_t smm = (size_t)3 * ma.P * bt * sizeof(V);
        if (smm > kSmemCap) {
            nm_set_error("padded length %d too long for the middle pass", ma.P);
            return NM_EUNSUPPORTED;
        }
        NM_TRY(set_smem(k_mid<T, PR>, smm));
        const dim3 gm((g.C1p + bt - 1) / bt, ma.n_fixed);
        {
            NmLaunchScope sc(mesh, NM_K_MID, st);
            k_mid<T, PR><<<gm, kThreads, smm, st>>>(midbuf, (const T *)mesh->Nhat, g, ma, bt, *mplan, mtw,
                                                kline, mesh->kmap_y, mesh->pos_y);
        }

    }
    if (g.N3 > 1) {
        int bt = Tile<T>::lines_y;
        while ((size_t)g.P2 * bt * sizeof(V) > kSmemCap && bt > 1) bt >>= 1;
        const size_t smy = (size_t)g.P2 * bt * sizeof(V);
        const dim3 gy((g.C1p + bt - 1) / bt, g.N3, 3);
        {
            NmLaunchScope sc(mesh, NM_K_Y_INV, st);
            k_lines<T, true, PR><<<gy, kThreads, smy, st>>>(B, A, g, bt, mesh->plan_y, (const V *)mesh->tw_y);
        }

    }
    {
        NmLaunchScope sc(mesh, NM_K_X_INV, st);
        if (rx2) {
            NM_TRY(set_smem(k_x_inv<T, 2, PR>, smx));
            k_x_inv<T, 2, PR><<<gx, kThreads, smx, st>>>(A, Hc_out, g, mesh->plan_x, (const V *)mesh->tw_x,
                                                    (const V *)mesh->tw_x2, mesh->pos_x);
        } else {
            NM_TRY(set_smem(k_x_inv<T, kRowsX, PR>, smx));
            k_x_inv<T, kRowsX, PR><<<gx, kThreads, smx, st>>>(A, Hc_out, g, mesh->plan_x, (const V *)mesh->tw_x,
                                                         (const V *)mesh->tw_x2, mesh->pos_x);
        }
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template nm_status nm_demag_conv<float>(nm_mesh *, const float *, float *, cudaStream_t);
template nm_status nm_demag_conv<double>(nm_mesh *, const double *, double *, cudaStream_t);
