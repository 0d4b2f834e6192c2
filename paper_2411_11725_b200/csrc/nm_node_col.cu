// Column-marching node kernel: a5-a11 of the hot path for uniform A and Ku.
//
// Same separable operators as k_node_sep (nm_local.cu):
//     (A v)_i = [i>0] (v_i - v_{i-1}) + [i<N] (v_i - v_{i+1})                 stiffness, K1
//     (B v)_i = [i>0] (v_i/3 + v_{i-1}/6) + [i<N] (v_i/3 + v_{i+1}/6)         mass, M1
//     E_n   = dx^-2 (Bz By Ax m) + dy^-2 (Bz Ay Bx m) + dz^-2 (Az By Bx m)    (Eqs. 17-22, reading C2)
//     H^ex  = -(16 A / (mu0 (S Ms)_n)) E_n,   H^an = (16 Ku / (mu0 (S Ms)_n)) (Bz By Bx (m.k)) k
//     H^d_n = S(Ms o H^cell)_n / (S Ms)_n                                     (reading C5)
// followed by the LLG products (Eq. 1), the Runge-Kutta stage combination (a10) or the adjoint
// products (a11, reading C7).
//
// What differs is how the SM is fed.  A CTA owns RY whole node rows (all of x: one thread per
// node column i1, so every global and shared access of a warp is a contiguous row segment) and
// marches along z.  Whole rows are contiguous in memory, so a plane's tile -- RY + 2 node rows of
// each component of m, RY + 1 cell rows of each component of H^cell (and of Ms) -- is a handful
// of contiguous ranges that cp.async (zero-filling what lies outside the mesh) streams into a
// ring of CS stages, CS - 1 planes ahead of the arithmetic: the loads of later planes are in
// flight while the current one is combined, one CTA barrier per plane.  Each thread keeps the x
// operators of a row in registers and reuses them for the RY rows it owns.  The epilogue is
// compiled per mode (template), so a stage launch carries no mode branches.
#include "nm_local.cuh"

namespace {

template <typename T> __device__ __forceinline__ T rsqrt_c(T v);
template <> __device__ __forceinline__ float rsqrt_c<float>(float v) { return 1.0f / sqrtf(v); }
template <> __device__ __forceinline__ double rsqrt_c<double>(double v) { return 1.0 / sqrt(v); }
template <typename T> __device__ __forceinline__ T abs_c(T v) { return v < 0 ? -v : v; }
template <typename T> __device__ __forceinline__ T max_c(T a, T b) { return a > b ? a : b; }

template <typename T> __device__ __forceinline__ void cross_c(const T *a, const T *b, T *c)
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// one element global -> shared, or zeros when !ok (src-size 0: nothing is read)
template <typename T> __device__ __forceinline__ void cp_elem(T *dst, const T *src, bool ok)
{
    const int sz = ok ? (int)sizeof(T) : 0;
    if (sizeof(T) == 4)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(smem_addr(dst)), "l"(src), "r"(sz) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_addr(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_16(void *dst, const void *src, bool ok)
{
    const int sz = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_addr(dst)), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ double block_sum_c(double v, int nthreads)
{
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = l < (nthreads + 31) / 32 ? red[l] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
    }
    return r;   // valid in thread 0
}

// modes of the compiled epilogues: the NmLocalMode values, with the Runge-Kutta stage split by the
// number of earlier derivatives it combines (0: first stages of RK4; 3: last stage of RK4; else a loop)
enum { CM_H = 0, CM_RHS, CM_RK0, CM_RK3, CM_RKN, CM_ADJ1, CM_ADJ2, CM_COUNT };

// a9-a11 on one node.  mc = fld_n, sms = (S Ms)_n.
template <typename T, int CM>
__device__ __forceinline__ void epilogue_c(const NmLocalArgs<T> &a, long long n, long long nn, const T *mc,
                                           const T *H, T sms, double &err2)
{
    if (CM == CM_H) {
        a.out[n] = H[0]; a.out[nn + n] = H[1]; a.out[2 * nn + n] = H[2];
        return;
    }
    if (CM == CM_ADJ2) {
#pragma unroll
        for (int j = 0; j < 3; ++j) a.dadt[j * nn + n] = -(a.dadt[j * nn + n] + sms * H[j]);
        return;
    }
    T mxH[3], mxmxH[3], f[3];
    cross_c(mc, H, mxH);
    cross_c(mc, mxH, mxmxH);
#pragma unroll
    for (int j = 0; j < 3; ++j) f[j] = -a.gp * mxH[j] - a.agp * mxmxH[j];
    if (CM == CM_RHS) {
        a.out[n] = f[0]; a.out[nn + n] = f[1]; a.out[2 * nn + n] = f[2];
    } else if (CM == CM_RK0 || CM == CM_RK3 || CM == CM_RKN) {
        const NmRkArgs<T> &r = a.rk;
        T y0[3], acc[3], ea[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            y0[j] = r.y0[j * nn + n];
            acc[j] = r.cself * f[j];
            ea[j] = r.eself * f[j];
        }
        if (CM == CM_RK3) {
#pragma unroll
            for (int q = 0; q < 3; ++q)
#pragma unroll
                for (int j = 0; j < 3; ++j) acc[j] += r.cprev[q] * r.kprev[q][j * nn + n];
        } else if (CM == CM_RKN) {
            for (int q = 0; q < r.nprev; ++q) {
                const T *kp = r.kprev[q] + n;
                const T cq = r.cprev[q], eq = r.eprev[q];
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    const T kv = kp[j * nn];
                    acc[j] += cq * kv;
                    ea[j] += eq * kv;
                }
            }
        }
        if (r.kstore) {
            r.kstore[n] = f[0]; r.kstore[nn + n] = f[1]; r.kstore[2 * nn + n] = f[2];
        }
        if (r.ynext) {
            T y[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) y[j] = y0[j] + r.dt * acc[j];
            if (r.renorm) {
                const T inv = rsqrt_c<T>(y[0] * y[0] + y[1] * y[1] + y[2] * y[2]);
                y[0] *= inv; y[1] *= inv; y[2] *= inv;
            }
            r.ynext[n] = y[0]; r.ynext[nn + n] = y[1]; r.ynext[2 * nn + n] = y[2];
        }
        if (CM == CM_RKN && r.want_err) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T sc = r.atol + r.rtol * max_c(abs_c(y0[j]), abs_c(mc[j]));
                const double q = (double)(r.dt * ea[j] / sc);
                err2 += q * q;
            }
        }
    } else {   // CM_ADJ1
        if (a.out) {
            a.out[n] = f[0]; a.out[nn + n] = f[1]; a.out[2 * nn + n] = f[2];
        }
        const T av[3] = {a.adj[n], a.adj[nn + n], a.adj[2 * nn + n]};
        T mxa[3], mxmxa[3], Hxa[3], b[3];
        cross_c(mc, av, mxa);
        cross_c(mc, mxa, mxmxa);
        cross_c(H, av, Hxa);
        const T mH = mc[0] * H[0] + mc[1] * H[1] + mc[2] * H[2];
        const T am = av[0] * mc[0] + av[1] * mc[1] + av[2] * mc[2];
        const T aH = av[0] * H[0] + av[1] * H[1] + av[2] * H[2];
        const T invS = sms > 0 ? (T)1 / sms : (T)0;
        T bH = 0;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            b[j] = a.gp * mxa[j] - a.agp * mxmxa[j];
            const T d = -a.gp * Hxa[j] - a.agp * (mH * av[j] + am * H[j] - (T)2 * aH * mc[j]);
            a.dadt[j * nn + n] = d;
            a.Q[j * nn + n] = b[j] * invS;
            bH += b[j] * H[j];
        }
        a.W[n] = bH * invS;
    }
}

// Tile geometry (host and device agree through this struct).  Per stage and component:
//   m tile     [PAD][(RY + 2) n1][tail]   node rows r0 - 1 .. r0 + RY, flattened (pitch n1)
//   cell tile  [PAD][(RY + 1) N1][tail]   cell rows r0 - 1 .. r0 + RY - 1 (pitch N1); 3 of H^cell (+ 1 of Ms)
// PAD elements in front absorb the index -1 of the first column, the tail the index +1 of the last.
struct ColGeom {
    int mpitch, cpitch;     // elements per component tile
    int ncell;              // cell tiles per stage: 0 (no demag), 3 (uniform Ms) or 4
    int stage;              // elements per stage
    int cvec;               // 1: cell rows are copied in 16-byte pieces
};
constexpr int CPAD = 4;

template <typename T, int RY> __host__ __device__ inline ColGeom col_geom(const NmGeom &g, bool has_hc, bool uni_ms)
{
    ColGeom c;
    const int blk = ((g.n1 + 31) / 32) * 32;
    c.mpitch = ((CPAD + (RY + 2) * g.n1 + (blk - g.n1) + 2 + 3) / 4) * 4;
    c.cpitch = ((CPAD + (RY + 1) * g.N1 + (blk - g.N1) + 2 + 3) / 4) * 4;
    c.ncell = has_hc ? (uni_ms ? 3 : 4) : 0;
    c.stage = 3 * c.mpitch + c.ncell * c.cpitch;
    c.cvec = ((g.N1 * sizeof(T)) % 16 == 0) ? 1 : 0;
    return c;
}

template <typename T, int RY, int CS, int CM, bool UNI_MS, int MAXT>
__global__ void __launch_bounds__(MAXT, sizeof(T) == 8 ? 1 : 2) k_node_col(const NmLocalArgs<T> a, int zchunk)
{
    extern __shared__ __align__(16) unsigned char col_smem[];
    T *sm = reinterpret_cast<T *>(col_smem);
    const NmGeom &g = a.g;
    const int n1 = g.n1, N1 = g.N1;
    const bool has_hc = a.Hc != nullptr;
    const ColGeom cg = col_geom<T, RY>(g, has_hc, UNI_MS);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int i1 = tid;
    const int r0 = blockIdx.x * RY;                       // first node row of the CTA
    const int z0 = blockIdx.y * zchunk, z1 = min(z0 + zchunk, g.n3);
    const long long pl = (long long)n1 * g.n2, nn = g.nodes;
    const long long cpl = (long long)N1 * g.N2;
    const bool live = i1 < n1;

    // the pads are never written by the copies: make them finite once
    for (int q = tid; q < CS * cg.stage; q += nthr) sm[q] = (T)0;
    __syncthreads();

    // rows of the tiles that exist in the mesh: node rows r0-1+r, r in [mlo, mhi); cell rows r0-1+r, r in [clo, chi)
    const int mlo = r0 == 0 ? 1 : 0, mhi = min(RY + 2, g.n2 - (r0 - 1));
    const int clo = mlo, chi = min(RY + 1, g.N2 - (r0 - 1));
    const int mlen = (RY + 2) * n1, clen = (RY + 1) * N1;

    auto issue = [&](int k, int slot) {
        T *st = sm + slot * cg.stage;
        const bool mv = k >= 0 && k < g.n3;
        {
            const T *src = a.fld + ((long long)k * g.n2 + (r0 - 1)) * n1;
            for (int e = tid; e < mlen; e += nthr) {
                const bool ok = mv && e >= mlo * n1 && e < mhi * n1;
                const T *s = ok ? src + e : a.fld;
                T *d = st + CPAD + e;
#pragma unroll
                for (int j = 0; j < 3; ++j) cp_elem<T>(d + j * cg.mpitch, s + j * nn, ok);
            }
        }
        if (has_hc) {
            const bool cv = k - 1 >= 0 && k - 1 < g.N3;
            const long long cbase = ((long long)(k - 1) * g.N2 + (r0 - 1)) * N1;
            T *dc = st + 3 * cg.mpitch + CPAD;
            if (cg.cvec) {
                constexpr int V = 16 / sizeof(T);
                for (int e = tid * V; e < clen; e += nthr * V) {
                    const bool ok = cv && e >= clo * N1 && e < chi * N1;
                    const long long off = ok ? cbase + e : 0;
#pragma unroll
                    for (int j = 0; j < 3; ++j) cp_16(dc + j * cg.cpitch + e, a.Hc + j * g.cells + off, ok);
                    if (!UNI_MS) cp_16(dc + 3 * cg.cpitch + e, a.Ms + off, ok);
                }
            } else {
                for (int e = tid; e < clen; e += nthr) {
                    const bool ok = cv && e >= clo * N1 && e < chi * N1;
                    const long long off = ok ? cbase + e : 0;
#pragma unroll
                    for (int j = 0; j < 3; ++j) cp_elem<T>(dc + j * cg.cpitch + e, a.Hc + j * g.cells + off, ok);
                    if (!UNI_MS) cp_elem<T>(dc + 3 * cg.cpitch + e, a.Ms + off, ok);
                }
            }
        }
    };

    // 1-D coefficients of this node column and of the RY rows
    const T third = (T)(1.0 / 3.0), sixth = (T)(1.0 / 6.0);
    const T eL = i1 > 0 ? (T)1 : (T)0, eR = i1 < N1 ? (T)1 : (T)0;
    const T bx0 = (eL + eR) * third, bxL = eL * sixth, bxR = eR * sixth;
    T fL[RY], fR[RY];
    bool rowlive[RY];
#pragma unroll
    for (int ry = 0; ry < RY; ++ry) {
        const int i2 = r0 + ry;
        fL[ry] = i2 > 0 ? (T)1 : (T)0;
        fR[ry] = i2 < g.N2 ? (T)1 : (T)0;
        rowlive[ry] = live && i2 < g.n2;
    }

    T Um[RY][3], U0[RY][3], Wm[RY][3], W0[RY][3], T0[RY][3], mc0[RY][3];
#pragma unroll
    for (int ry = 0; ry < RY; ++ry)
#pragma unroll
        for (int j = 0; j < 3; ++j) Um[ry][j] = U0[ry][j] = Wm[ry][j] = W0[ry][j] = T0[ry][j] = mc0[ry][j] = (T)0;
    double err2 = 0.0;

    const int kstart = max(z0 - 1, 0), kend = z1;         // kend may be n3 (no such plane: zeros)
#pragma unroll
    for (int s = 0; s < CS - 1; ++s) {
        if (kstart + s <= kend) issue(kstart + s, s);
        cp_commit();
    }
    int slot = 0;
    for (int k = kstart; k <= kend; ++k) {
        cp_wait<CS - 2>();
        __syncthreads();
        {
            const int kn = k + CS - 1;
            int sn = slot + CS - 1;
            if (sn >= CS) sn -= CS;
            if (kn <= kend) issue(kn, sn);
            cp_commit();
        }
        const T *st = sm + slot * cg.stage;
        T Up[RY][3], Wp[RY][3], Tn[RY][3], mcn[RY][3];
        if (live) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T *t = st + j * cg.mpitch + CPAD + i1;
                T P[RY + 2], Q[RY + 2];
#pragma unroll
                for (int r = 0; r < RY + 2; ++r) {
                    const T *row = t + r * n1;
                    const T l = row[-1], c = row[0], rr = row[1];
                    Q[r] = eL * (c - l) + eR * (c - rr);
                    P[r] = bx0 * c + bxL * l + bxR * rr;
                    if (r >= 1 && r <= RY) mcn[r - 1][j] = c;
                }
#pragma unroll
                for (int ry = 0; ry < RY; ++ry) {
                    const T by0 = (fL[ry] + fR[ry]) * third, byL = fL[ry] * sixth, byR = fR[ry] * sixth;
                    const T AyP = fL[ry] * (P[ry + 1] - P[ry]) + fR[ry] * (P[ry + 1] - P[ry + 2]);
                    const T ByQ = by0 * Q[ry + 1] + byL * Q[ry] + byR * Q[ry + 2];
                    Wp[ry][j] = by0 * P[ry + 1] + byL * P[ry] + byR * P[ry + 2];
                    Up[ry][j] = a.idx2[0] * ByQ + a.idx2[1] * AyP;
                }
            }
            if (has_hc) {
                const T *cb = st + 3 * cg.mpitch + CPAD + i1;
                T wl_[RY + 1], wr_[RY + 1];                // x weights of the two cells of a row (eL, eR, times Ms)
#pragma unroll
                for (int cr = 0; cr < RY + 1; ++cr) {
                    if (UNI_MS) { wl_[cr] = eL; wr_[cr] = eR; }
                    else {
                        const T *mrow = cb + 3 * cg.cpitch + cr * N1;
                        wl_[cr] = eL * mrow[-1];
                        wr_[cr] = eR * mrow[0];
                    }
                }
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    T X[RY + 1];
#pragma unroll
                    for (int cr = 0; cr < RY + 1; ++cr) {
                        const T *crow = cb + j * cg.cpitch + cr * N1;
                        X[cr] = wl_[cr] * crow[-1] + wr_[cr] * crow[0];
                    }
#pragma unroll
                    for (int ry = 0; ry < RY; ++ry) Tn[ry][j] = fL[ry] * X[ry] + fR[ry] * X[ry + 1];
                }
            } else {
#pragma unroll
                for (int ry = 0; ry < RY; ++ry) Tn[ry][0] = Tn[ry][1] = Tn[ry][2] = (T)0;
            }
        }
        const int z = k - 1;
        if (z >= z0 && z < z1) {
            const T gL = z > 0 ? (T)1 : (T)0, gR = z < g.N3 ? (T)1 : (T)0;
            const T bz0 = (gL + gR) * third, bzL = gL * sixth, bzR = gR * sixth;
#pragma unroll
            for (int ry = 0; ry < RY; ++ry) {
                if (!rowlive[ry]) continue;
                const long long n = (long long)z * pl + (long long)(r0 + ry) * n1 + i1;
                const T sms = UNI_MS ? a.ms_uni * (eL + eR) * (fL[ry] + fR[ry]) * (gL + gR) : a.sMs[n];
                T H[3] = {0, 0, 0};
                if (sms > 0) {
                    const T inv = (T)1 / sms;
                    T an = 0;
#pragma unroll
                    for (int j = 0; j < 3; ++j) an += a.kax[j] * (bz0 * W0[ry][j] + bzL * Wm[ry][j] + bzR * Wp[ry][j]);
                    const T dsc = UNI_MS ? a.ms_uni * inv : inv;       // demag average weight
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        const T E = (bz0 * U0[ry][j] + bzL * Um[ry][j] + bzR * Up[ry][j]) +
                                    a.idx2[2] * (gL * (W0[ry][j] - Wm[ry][j]) + gR * (W0[ry][j] - Wp[ry][j]));
                        T hv = (a.cku * an * a.kax[j] - a.cex * E) * inv + (T0[ry][j] + Tn[ry][j]) * dsc;
                        if (a.terms & NM_TERM_ZEEMAN) hv += a.hu[j];
                        H[j] = hv;
                    }
                }
                epilogue_c<T, CM>(a, n, nn, mc0[ry], H, sms, err2);
            }
        }
#pragma unroll
        for (int ry = 0; ry < RY; ++ry)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                Um[ry][j] = U0[ry][j]; U0[ry][j] = Up[ry][j];
                Wm[ry][j] = W0[ry][j]; W0[ry][j] = Wp[ry][j];
                T0[ry][j] = Tn[ry][j]; mc0[ry][j] = mcn[ry][j];
            }
        if (++slot == CS) slot = 0;
    }
    cp_wait<0>();
    if (CM == CM_RKN) {
        if (a.rk.want_err) {
            const double s = block_sum_c(err2, nthr);
            if (tid == 0) a.rk.partials[blockIdx.y * gridDim.x + blockIdx.x] = s;
        }
    }
}

constexpr int kRY = 2;
constexpr int kMaxT = 320;
template <typename T> struct ColStages { static constexpr int CS = sizeof(T) == 8 ? 3 : 4; };

inline int col_zchunk(const NmGeom &g) { return g.n3 <= 40 ? g.n3 : 32; }

template <typename T, int CM, bool UNI_MS>
nm_status launch_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    constexpr int CS = ColStages<T>::CS;
    const NmGeom &g = a.g;
    const ColGeom cg = col_geom<T, kRY>(g, a.Hc != nullptr, UNI_MS);
    const size_t bytes = (size_t)CS * cg.stage * sizeof(T);
    const int zchunk = col_zchunk(g);
    const dim3 grid((g.n2 + kRY - 1) / kRY, (g.n3 + zchunk - 1) / zchunk);
    const int threads = ((g.n1 + 31) / 32) * 32;
    auto kern = k_node_col<T, kRY, CS, CM, UNI_MS, kMaxT>;
    NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    mesh->last_partials = (int)(grid.x * grid.y);
    {
        NmLaunchScope sc(mesh, NM_K_NODE, st);
        kern<<<grid, threads, bytes, st>>>(a, zchunk);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T, bool UNI_MS> nm_status dispatch_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    switch (a.mode) {
    case NM_MODE_H: return launch_col<T, CM_H, UNI_MS>(mesh, a, st);
    case NM_MODE_RHS: return launch_col<T, CM_RHS, UNI_MS>(mesh, a, st);
    case NM_MODE_ADJ1: return launch_col<T, CM_ADJ1, UNI_MS>(mesh, a, st);
    case NM_MODE_ADJ2: return launch_col<T, CM_ADJ2, UNI_MS>(mesh, a, st);
    default:
        if (!a.rk.want_err && a.rk.nprev == 0) return launch_col<T, CM_RK0, UNI_MS>(mesh, a, st);
        if (!a.rk.want_err && a.rk.nprev == 3) return launch_col<T, CM_RK3, UNI_MS>(mesh, a, st);
        return launch_col<T, CM_RKN, UNI_MS>(mesh, a, st);
    }
}

} // namespace

// Eligibility: the separable operators (uniform A, Ku; no nodal Zeeman arrays -- decided by the
// caller), a thread per node column, and a ring of stages that fits the shared memory of an SM.
template <typename T> bool nm_node_col_ok(const nm_mesh *mesh, const NmLocalArgs<T> &a)
{
    const NmGeom &g = a.g;
    if (g.n1 < 96 || g.n1 > kMaxT) return false;
    const ColGeom cg = col_geom<T, kRY>(g, a.Hc != nullptr, a.ms_uni > 0);
    const size_t bytes = (size_t)ColStages<T>::CS * cg.stage * sizeof(T);
    (void)mesh;
    if (cg.cvec && a.Hc && ((((uintptr_t)a.Hc) | ((uintptr_t)a.Ms)) & 15)) return false;   // 16-byte cell copies
    return bytes <= (sizeof(T) == 8 ? 200u : 110u) * 1024u;
}

template <typename T> nm_status nm_launch_node_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    return a.ms_uni > 0 ? dispatch_col<T, true>(mesh, a, st) : dispatch_col<T, false>(mesh, a, st);
}

int nm_node_col_blocks(const NmGeom &g)
{
    const int zchunk = col_zchunk(g);
    return ((g.n2 + kRY - 1) / kRY) * ((g.n3 + zchunk - 1) / zchunk);
}

template bool nm_node_col_ok<float>(const nm_mesh *, const NmLocalArgs<float> &);
template bool nm_node_col_ok<double>(const nm_mesh *, const NmLocalArgs<double> &);
template nm_status nm_launch_node_col<float>(nm_mesh *, const NmLocalArgs<float> &, cudaStream_t);
template nm_status nm_launch_node_col<double>(nm_mesh *, const NmLocalArgs<double> &, cudaStream_t);
