// Node and cell kernels: a5-a11 of the hot path.
//
// One thread per node evaluates, in one pass over the 27-node neighbourhood and the 8 adjacent
// cells,
//   exchange    H = -(1/L_n) sum_{c∋n} 2 A_c sum_i' K[i,i'] m_{c+i'}        (Eqs. 3, 17-22; C3)
//   anisotropy  H = +(1/L_n) sum_{c∋n} 2 Ku_c sum_i' M[i,i'] (m_{c+i'}.k) k  (reading C3(i))
//   Zeeman      H = (mu0/L_n) sum_{c∋n} Ms_c sum_i' M[i,i'] Hext_{c+i'}      (Eq. 21; C3(ii))
//   demag       H = sum_{c∋n} Ms_c Hcell_c / sum_{c∋n} Ms_c                  (C5)
// with L_n = mu0 (V/8) sum_{c∋n} Ms_c (Eq. 22), then the LLG cross products of Eq. (1) and the
// Runge-Kutta stage combination (a10) or the adjoint products of reading C7 (a11).
//
// The element matrices only depend on which coordinates of the two vertices differ, so the
// cell loop of Eqs. (19)-(20) is regrouped by neighbour offset delta in {-1,0,1}^3: the weight of
// m_{n+delta} is K[e(delta)] times the sum of 2 A_c over the cells that contain both nodes.  The
// exchange term is accumulated in difference form sum w (m_{n+delta} - m_n) (rows of K sum to
// zero), which keeps fp32 exact for smooth m.
#include "nm_local.cuh"

namespace {

constexpr int kBlock = 256;

template <typename T> __device__ __forceinline__ T rsqrt_t(T v);
template <> __device__ __forceinline__ float rsqrt_t<float>(float v) { return 1.0f / sqrtf(v); }
template <> __device__ __forceinline__ double rsqrt_t<double>(double v) { return 1.0 / sqrt(v); }

template <typename T> __device__ __forceinline__ T abs_t(T v) { return v < 0 ? -v : v; }
template <typename T> __device__ __forceinline__ T max_t(T a, T b) { return a > b ? a : b; }

template <typename T>
__device__ __forceinline__ void cross3(const T *a, const T *b, T *c)
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int t = threadIdx.y * blockDim.x + threadIdx.x;
    const int w = t >> 5, l = t & 31;
    if (l == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = l < (blockDim.x * blockDim.y + 31) / 32 ? red[l] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
    }
    return r;   // valid in thread (0, 0)
}

// a9-a11 on one node: what to do with H_n (modes of nm_local.cuh).  mc = fld_n, sms = (S Ms)_n.
template <typename T>
__device__ __forceinline__ void node_epilogue(const NmLocalArgs<T> &a, long long n, long long nn,
                                              const T *mc, const T *H, T sms, double &err2)
{
    if (a.mode == NM_MODE_H) {
        a.out[n] = H[0]; a.out[nn + n] = H[1]; a.out[2 * nn + n] = H[2];
    } else if (a.mode == NM_MODE_ADJ2) {
        // dadt = -(d + (S Ms) Hlin(q));  fld = q, H = Hlin(q)
#pragma unroll
        for (int j = 0; j < 3; ++j) a.dadt[j * nn + n] = -(a.dadt[j * nn + n] + sms * H[j]);
    } else {
        T mxH[3], mxmxH[3], f[3];
        cross3(mc, H, mxH);
        cross3(mc, mxH, mxmxH);
#pragma unroll
        for (int j = 0; j < 3; ++j) f[j] = -a.gp * mxH[j] - a.agp * mxmxH[j];
        if (a.mode == NM_MODE_RHS) {
            a.out[n] = f[0]; a.out[nn + n] = f[1]; a.out[2 * nn + n] = f[2];
        } else if (a.mode == NM_MODE_RK) {
            const NmRkArgs<T> &r = a.rk;
            if (r.kstore) {
                r.kstore[n] = f[0]; r.kstore[nn + n] = f[1]; r.kstore[2 * nn + n] = f[2];
            }
            T y0[3], y[3], er[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                y0[j] = r.y0[j * nn + n];
                T acc = r.cself * f[j];
                T ea = r.eself * f[j];
                for (int q = 0; q < r.nprev; ++q) {
                    const T kp = r.kprev[q][j * nn + n];
                    acc += r.cprev[q] * kp;
                    ea += r.eprev[q] * kp;
                }
                y[j] = y0[j] + r.dt * acc;
                if (r.nstate == 2)
                    y[j] = r.bs[0] * y0[j] + r.bs[1] * r.sprev[0][j * nn + n] + r.bs[2] * r.sprev[1][j * nn + n] +
                           r.bs[3] * mc[j] + r.dt * acc;
                er[j] = r.dt * ea;
            }
            if (r.ynext) {
                if (r.renorm) {
                    const T n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
                    const T inv = n2 > (T)0 ? rsqrt_t<T>(n2) : (T)0;   // a zero vector (vacuum node) stays zero
                    y[0] *= inv; y[1] *= inv; y[2] *= inv;
                }
                r.ynext[n] = y[0]; r.ynext[nn + n] = y[1]; r.ynext[2 * nn + n] = y[2];
            }
            if (r.want_err) {
                // last Dormand-Prince stage: fld = y5 (un-normalised), y0 = start of step
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    const T sc = r.atol + r.rtol * max_t(abs_t(y0[j]), abs_t(mc[j]));
                    const double q = (double)(er[j] / sc);
                    err2 += q * q;
                }
            }
        } else {   // NM_MODE_ADJ1
            if (a.out) {
                a.out[n] = f[0]; a.out[nn + n] = f[1]; a.out[2 * nn + n] = f[2];
            }
            const T av[3] = {a.adj[n], a.adj[nn + n], a.adj[2 * nn + n]};
            T mxa[3], mxmxa[3], Hxa[3], b[3];
            cross3(mc, av, mxa);
            cross3(mc, mxa, mxmxa);
            cross3(H, av, Hxa);
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
}

// EXTRA = false: exchange + demag + uniform Zeeman only (no anisotropy, no nodal Zeeman arrays).
// Grid: x = blocks of kBlock nodes of one z plane (flattened i2*n1 + i1), y = i3.
// A neighbour or cell that does not exist is read at a clamped (valid) address and only ever
// multiplied by a zero coefficient, so the kernel has no per-neighbour branches.
template <typename T, bool EXTRA>
__global__ void __launch_bounds__(kBlock) k_node(const NmLocalArgs<T> a)
{
    const NmGeom &g = a.g;
    const int pl = g.n1 * g.n2;
    const int p = blockIdx.x * kBlock + threadIdx.x;
    const int i3 = blockIdx.y;
    const bool live = p < pl;
    double err2 = 0.0;
    if (live) {
        const int i2 = p / g.n1, i1 = p - i2 * g.n1;
        const long long nn = g.nodes;
        const long long n = (long long)i3 * pl + p;
        const int ox[3] = {i1 > 0 ? -1 : 0, 0, i1 < g.N1 ? 1 : 0};
        // strides g.ys / g.zs: 0 along an axis the basis does not vary in (the +1 neighbour is the node itself)
        const int oy[3] = {i2 > 0 ? -g.ys : 0, 0, i2 < g.N2 ? g.ys : 0};
        const int oz[3] = {i3 > 0 ? -g.zs : 0, 0, i3 < g.N3 ? g.zs : 0};
        // the 8 adjacent cells (bit 0: x, 1: y, 2: z; 0 = lower side)
        const bool vx[2] = {i1 > 0, i1 < g.N1}, vy[2] = {i2 > 0, i2 < g.N2}, vz[2] = {i3 > 0, i3 < g.N3};
        const int cx[2] = {i1 > 0 ? i1 - 1 : 0, i1 < g.N1 ? i1 : g.N1 - 1};
        const int cy[2] = {i2 > 0 ? i2 - 1 : 0, i2 < g.N2 ? i2 : g.N2 - 1};
        const int cz[2] = {i3 > 0 ? i3 - 1 : 0, i3 < g.N3 ? i3 : g.N3 - 1};
        const bool ex_on = (a.terms & NM_TERM_EXCHANGE) != 0;
        T cA[8], cK[8], cM[8];
        T hd[3] = {0, 0, 0};
        T sms = 0;
#pragma unroll
        for (int ci = 0; ci < 8; ++ci) {
            const int bx = ci & 1, by = (ci >> 1) & 1, bz = ci >> 2;
            const long long c = ((long long)cz[bz] * g.N2 + cy[by]) * g.N1 + cx[bx];
            const bool ok = vx[bx] && vy[by] && vz[bz];
            const T ms = ok ? a.Ms[c] : (T)0;
            cM[ci] = ms;
            cA[ci] = (ok && ex_on) ? (T)2 * a.A[c] : (T)0;
            if (EXTRA) cK[ci] = (ok && (a.terms & NM_TERM_ANISO)) ? (T)2 * a.Ku[c] : (T)0;
            if (a.Hc) {
                hd[0] += ms * a.Hc[c];
                hd[1] += ms * a.Hc[g.cells + c];
                hd[2] += ms * a.Hc[2 * g.cells + c];
            }
            sms += ms;
        }
        const T *f0 = a.fld + n, *f1 = f0 + nn, *f2 = f1 + nn;
        const T mc[3] = {f0[0], f1[0], f2[0]};
        const bool zee_on = (a.terms & NM_TERM_ZEEMAN) != 0;
        const bool zee_nodal = EXTRA && zee_on && (a.h_static || a.h_pulse);
        T ex[3] = {0, 0, 0}, ze[3] = {0, 0, 0};
        T an = 0;
#pragma unroll
        for (int dz = -1; dz <= 1; ++dz)
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) {
                    const int e = (dx != 0) | ((dy != 0) << 1) | ((dz != 0) << 2);
                    if (e == 0 && !EXTRA) continue;
                    // cells that contain both n and n + delta
                    T sA = 0, sK = 0, sM = 0;
#pragma unroll
                    for (int ci = 0; ci < 8; ++ci) {
                        const int bx = ci & 1, by = (ci >> 1) & 1, bz = ci >> 2;
                        const bool in = (dx == 0 || bx == (dx + 1) / 2) && (dy == 0 || by == (dy + 1) / 2) &&
                                        (dz == 0 || bz == (dz + 1) / 2);
                        if (in) {
                            sA += cA[ci];
                            if (EXTRA) { sK += cK[ci]; sM += cM[ci]; }
                        }
                    }
                    const int off = ox[dx + 1] + oy[dy + 1] + oz[dz + 1];
                    T mb[3];
                    if (e == 0) {
                        mb[0] = mc[0]; mb[1] = mc[1]; mb[2] = mc[2];
                    } else {
                        mb[0] = f0[off]; mb[1] = f1[off]; mb[2] = f2[off];
                        const T w = a.wK[e] * sA;
                        ex[0] += w * (mb[0] - mc[0]);
                        ex[1] += w * (mb[1] - mc[1]);
                        ex[2] += w * (mb[2] - mc[2]);
                    }
                    if (EXTRA) {
                        an += a.wM[e] * sK * (mb[0] * a.kax[0] + mb[1] * a.kax[1] + mb[2] * a.kax[2]);
                        if (zee_nodal) {
                            const T w = a.wM[e] * sM;
#pragma unroll
                            for (int j = 0; j < 3; ++j) {
                                T hv = 0;
                                if (a.h_static) hv += a.h_static[j * nn + n + off];
                                if (a.h_pulse) hv += a.amp * a.h_pulse[j * nn + n + off];
                                ze[j] += w * hv;
                            }
                        }
                    }
                }

        T H[3] = {0, 0, 0};
        if (sms > 0) {
            const T invL = (T)1 / (a.mu0V8 * sms);
            const T invS = (T)1 / sms;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                T hv = (a.kax[j] * an - ex[j]) * invL + hd[j] * invS;
                if (zee_on) hv += a.hu[j];
                if (zee_nodal) hv += a.mu0 * ze[j] * invL;
                if (a.hadd) hv += a.hadd[j * nn + n];
                H[j] = hv;
            }
        }

        node_epilogue<T>(a, n, nn, mc, H, sms, err2);
    }
    if (a.mode == NM_MODE_RK && a.rk.want_err) {
        const double s = block_sum(err2);
        if (threadIdx.x == 0) a.rk.partials[blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
}


// a8 with nodal external fields, separately from the other terms (they are linear in H_ext and do not
// involve m): Zs_n = (mu0 / L_n) sum_{c in n} Ms_c sum_{i'} M_{i,i'} H^ext_{c+i'}  (Eq. 21, reading
// C3(ii)), H^ext = h_static + amp h_pulse; 0 where (S Ms)_n = 0.  Lets meshes with uniform A and Ku keep
// the separable node kernels when the Zeeman field is a nodal array (config 3's stripe pulse).
// GRAD: the transpose of the same operator, for the gradient with respect to a nodal external field
// (SURVEY.md 8(f) row 2): with h := q = b / (S Ms),  out (+)= coef (-(8/V) sum_c Ms_c sum_i' M_{i,i'} q_{c+i'})
// = coef Z(b / L) = -coef (df/dh)^T a  (oracle/adjoint.py: adjoint_rhs_hnodal).
// A CTA owns a ZX x ZY patch of nodes of one plane: the field (h_static + amp h_pulse) of the patch, its halo and the
// two neighbouring planes goes through shared memory once, and the 27-point sums read it from there.
constexpr int ZX = 32, ZY = 8, ZPX = ZX + 2, ZPY = ZY + 2;
template <typename T, bool GRAD>
__global__ void __launch_bounds__(ZX * ZY) k_zeeman_smooth(const NmLocalArgs<T> a, T *__restrict__ Zs, T coef, int accumulate)
{
    __shared__ T sh[3][3][ZPY][ZPX];
    const NmGeom &g = a.g;
    const long long nn = g.nodes;
    const int x0 = blockIdx.x * ZX, y0 = blockIdx.y * ZY, i3 = blockIdx.z;
    // a thread fills (xx, yy) = (tx, ty) and, at the patch edges, (tx + ZX, .) for tx < 2 and (., ty + ZY) for ty < 2
    // along an axis the basis does not vary in, every neighbour is the node itself (strides g.ys / g.zs = 0)
    auto fill = [&](auto value) {
#pragma unroll
        for (int ry = 0; ry < 2; ++ry) {
            const int yy = threadIdx.y + ry * ZY;
            const int gy = g.ys ? y0 - 1 + yy : 0;
#pragma unroll
            for (int rx = 0; rx < 2; ++rx) {
                const int xx = threadIdx.x + rx * ZX;
                const int gx = x0 - 1 + xx;
                const bool mine = (!ry || threadIdx.y < 2) && (!rx || threadIdx.x < 2);
                const bool okxy = mine && gx >= 0 && gx < g.n1 && gy >= 0 && gy < g.n2;
#pragma unroll
                for (int dz = 0; dz < 3; ++dz) {
                    const int gz = g.zs ? i3 - 1 + dz : 0;
                    const bool ok = okxy && gz >= 0 && gz < g.n3;
                    const long long q = ok ? ((long long)gz * g.n2 + gy) * g.n1 + gx : 0;
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        const T v = value(j * nn + q);
                        if (mine) sh[j][dz][yy][xx] = ok ? v : (T)0;
                    }
                }
            }
        }
    };
    if (a.h_static && a.h_pulse) fill([&](long long q) { return a.h_static[q] + a.amp * a.h_pulse[q]; });
    else if (a.h_pulse) fill([&](long long q) { return a.amp * a.h_pulse[q]; });
    else if (a.h_static) fill([&](long long q) { return a.h_static[q]; });
    else fill([&](long long) { return (T)0; });
    __syncthreads();
    const int i1 = x0 + threadIdx.x, i2 = y0 + threadIdx.y;
    if (i1 >= g.n1 || i2 >= g.n2) return;
    const long long n = ((long long)i3 * g.n2 + i2) * g.n1 + i1;
    const bool vx[2] = {i1 > 0, i1 < g.N1}, vy[2] = {i2 > 0, i2 < g.N2}, vz[2] = {i3 > 0, i3 < g.N3};
    const int cx[2] = {i1 > 0 ? i1 - 1 : 0, i1 < g.N1 ? i1 : g.N1 - 1};
    const int cy[2] = {i2 > 0 ? i2 - 1 : 0, i2 < g.N2 ? i2 : g.N2 - 1};
    const int cz[2] = {i3 > 0 ? i3 - 1 : 0, i3 < g.N3 ? i3 : g.N3 - 1};
    T cM[8], sms = 0;
#pragma unroll
    for (int ci = 0; ci < 8; ++ci) {
        const int bx = ci & 1, by = (ci >> 1) & 1, bz = ci >> 2;
        const long long c = ((long long)cz[bz] * g.N2 + cy[by]) * g.N1 + cx[bx];
        cM[ci] = (vx[bx] && vy[by] && vz[bz]) ? a.Ms[c] : (T)0;
        sms += cM[ci];
    }
    // Ms summed over the cells that contain both n and n + delta (none: the neighbour does not exist), axis by axis:
    // offset -1 / +1 along an axis keeps the cells on that side, offset 0 keeps both
    T sx[3][2][2], sxy[3][3][2];
#pragma unroll
    for (int bz = 0; bz < 2; ++bz)
#pragma unroll
        for (int by = 0; by < 2; ++by) {
            const T lo = cM[by * 2 + bz * 4], hi = cM[1 + by * 2 + bz * 4];
            sx[0][by][bz] = lo; sx[1][by][bz] = lo + hi; sx[2][by][bz] = hi;
        }
#pragma unroll
    for (int dx = 0; dx < 3; ++dx)
#pragma unroll
        for (int bz = 0; bz < 2; ++bz) {
            sxy[dx][0][bz] = sx[dx][0][bz]; sxy[dx][1][bz] = sx[dx][0][bz] + sx[dx][1][bz]; sxy[dx][2][bz] = sx[dx][1][bz];
        }
    T ze[3] = {0, 0, 0};
#pragma unroll
    for (int dz = -1; dz <= 1; ++dz)
#pragma unroll
        for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
            for (int dx = -1; dx <= 1; ++dx) {
                const int e = (dx != 0) | ((dy != 0) << 1) | ((dz != 0) << 2);
                const T lo = sxy[dx + 1][dy + 1][0], hi = sxy[dx + 1][dy + 1][1];
                const T sM = dz < 0 ? lo : (dz > 0 ? hi : lo + hi);
                const T w = a.wM[e] * sM;
#pragma unroll
                for (int j = 0; j < 3; ++j) ze[j] += w * sh[j][dz + 1][threadIdx.y + 1 + dy][threadIdx.x + 1 + dx];
            }
    const T sc = sms > 0 ? a.mu0 / (a.mu0V8 * sms) : (T)0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        if (GRAD) {
            const T gv = -coef * (a.mu0 / a.mu0V8) * ze[j];
            Zs[j * nn + n] = accumulate ? Zs[j * nn + n] + gv : gv;
        } else {
            Zs[j * nn + n] = sc * ze[j] + (a.hadd ? a.hadd[j * nn + n] : (T)0);   // + the field of the further local terms
        }
    }
}

// q = b / (S Ms), b = g' m x a - alpha g' m x (m x a); 0 where (S Ms)_n = 0
template <typename T>
__global__ void k_bq(const T *__restrict__ m, const T *__restrict__ av, const T *__restrict__ sMs, long long nn, T gp, T agp,
                     T *__restrict__ Q)
{
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= nn) return;
    const T mm[3] = {m[n], m[nn + n], m[2 * nn + n]}, aa[3] = {av[n], av[nn + n], av[2 * nn + n]};
    const T mxa[3] = {mm[1] * aa[2] - mm[2] * aa[1], mm[2] * aa[0] - mm[0] * aa[2], mm[0] * aa[1] - mm[1] * aa[0]};
    const T mm2[3] = {mm[1] * mxa[2] - mm[2] * mxa[1], mm[2] * mxa[0] - mm[0] * mxa[2], mm[0] * mxa[1] - mm[1] * mxa[0]};
    const T s = sMs[n];
    const T inv = s > 0 ? (T)1 / s : (T)0;
#pragma unroll
    for (int j = 0; j < 3; ++j) Q[j * nn + n] = (gp * mxa[j] - agp * mm2[j]) * inv;
}

// -------------------------------------------------------------------------------------------------
// Separable node kernel for uniform A and Ku (scalars at nm_mesh_create), any Ms.
//
// With a cell-constant coefficient the assembled tensor-product element operators of Eqs. (19)-(20)
// factor into assembled 1-D operators along each axis (C2: K = V sum_d dx_d^-2 K1 (x) M1 (x) M1,
// M = V M1 (x) M1 (x) M1):
//     (A v)_i = [i>0] (v_i - v_{i-1}) + [i<N] (v_i - v_{i+1})                 stiffness, K1
//     (B v)_i = [i>0] (v_i/3 + v_{i-1}/6) + [i<N] (v_i/3 + v_{i+1}/6)         mass, M1
//     E_n   = dx^-2 (Bz By Ax m) + dy^-2 (Bz Ay Bx m) + dz^-2 (Az By Bx m)
//     H^ex  = -(16 A / (mu0 (S Ms)_n)) E_n,   H^an = (16 Ku / (mu0 (S Ms)_n)) (Bz By Bx (m.k)) k
// and the one-sided boundary stencils / reduced lumped mass of Eq. (22) come out of the [.] factors.
// A CTA owns an SX x SY patch of node columns and marches along z: per plane it stages the m tile
// (+1 halo) and the cell tile of H^cell in shared memory, forms the in-plane parts
//     U = dx^-2 By Ax m + dy^-2 Ay Bx m,   W = By Bx m,   T = sum over the 2x2 cells of w_c Hc_c
// and combines three consecutive planes in registers.  The next plane is prefetched into registers
// while the current one is being used (one barrier per plane).
constexpr int SX = 32, SY = 8;
constexpr int MP = SX + 2;              // m tile pitch
constexpr int MT = (SY + 2) * MP;       // m tile elements per component
constexpr int CPT = SX + 1;             // cell tile pitch
constexpr int CT = (SY + 1) * CPT;      // cell tile elements per component
constexpr int MR = (MT + SX * SY - 1) / (SX * SY);
constexpr int CR = (CT + SX * SY - 1) / (SX * SY);

template <typename T, bool UNI_MS>
__global__ void __launch_bounds__(SX * SY) k_node_sep(const NmLocalArgs<T> a, int zchunk)
{
    const NmGeom &g = a.g;
    __shared__ T s_m[2][3][MT];
    __shared__ T s_c[2][3][CT];
    const int tid = threadIdx.y * SX + threadIdx.x;
    const int x0 = blockIdx.x * SX, y0 = blockIdx.y * SY;
    const int i1 = x0 + threadIdx.x, i2 = y0 + threadIdx.y;
    const bool live = i1 < g.n1 && i2 < g.n2;
    const int z0 = blockIdx.z * zchunk;
    const int z1 = min(z0 + zchunk, g.n3);
    const long long pl = (long long)g.n1 * g.n2, nn = g.nodes;
    const long long cpl = (long long)g.N1 * g.N2;
    const bool has_hc = a.Hc != nullptr;

    // global offsets of this thread's tile elements (-1: outside the mesh -> 0)
    int m_off[MR], c_off[CR];
#pragma unroll
    for (int r = 0; r < MR; ++r) {
        const int idx = tid + r * SX * SY;
        const int ly = idx / MP, lx = idx - ly * MP;
        const int gx = x0 - 1 + lx, gy = y0 - 1 + ly;
        m_off[r] = (idx < MT && gx >= 0 && gx < g.n1 && gy >= 0 && gy < g.n2) ? gy * g.n1 + gx : -1;
    }
#pragma unroll
    for (int r = 0; r < CR; ++r) {
        const int idx = tid + r * SX * SY;
        const int ly = idx / CPT, lx = idx - ly * CPT;
        const int gx = x0 - 1 + lx, gy = y0 - 1 + ly;
        c_off[r] = (idx < CT && gx >= 0 && gx < g.N1 && gy >= 0 && gy < g.N2) ? gy * g.N1 + gx : -1;
    }
    // 1-D coefficients of this node column
    const T eL = i1 > 0 ? (T)1 : (T)0, eR = i1 < g.N1 ? (T)1 : (T)0;
    const T fL = i2 > 0 ? (T)1 : (T)0, fR = i2 < g.N2 ? (T)1 : (T)0;
    const T third = (T)(1.0 / 3.0), sixth = (T)(1.0 / 6.0);
    const T bx0 = (eL + eR) * third, bxL = eL * sixth, bxR = eR * sixth;
    const T by0 = (fL + fR) * third, byL = fL * sixth, byR = fR * sixth;
    const T cxy = (eL + eR) * (fL + fR);            // adjacent cells per plane of cells

    T pm[MR][3], pc[CR][3];
    auto fetch = [&](int k) {
        // m plane k (node plane) and cell plane k - 1
        const bool mv = k >= 0 && k < g.n3;
        const bool cv = has_hc && k - 1 >= 0 && k - 1 < g.N3;
#pragma unroll
        for (int r = 0; r < MR; ++r)
#pragma unroll
            for (int j = 0; j < 3; ++j)
                pm[r][j] = (mv && m_off[r] >= 0) ? a.fld[j * nn + (long long)k * pl + m_off[r]] : (T)0;
#pragma unroll
        for (int r = 0; r < CR; ++r) {
            const bool ok = cv && c_off[r] >= 0;
            const long long c = (long long)(k - 1) * cpl + c_off[r];
            if (UNI_MS) {
#pragma unroll
                for (int j = 0; j < 3; ++j) pc[r][j] = ok ? a.Hc[j * g.cells + c] : (T)0;
            } else {
                const T ms = ok ? a.Ms[c] : (T)0;
#pragma unroll
                for (int j = 0; j < 3; ++j) pc[r][j] = ok ? ms * a.Hc[j * g.cells + c] : (T)0;
            }
        }
    };
    auto stash = [&](int b) {
#pragma unroll
        for (int r = 0; r < MR; ++r) {
            const int idx = tid + r * SX * SY;
            if (idx < MT) {
#pragma unroll
                for (int j = 0; j < 3; ++j) s_m[b][j][idx] = pm[r][j];
            }
        }
#pragma unroll
        for (int r = 0; r < CR; ++r) {
            const int idx = tid + r * SX * SY;
            if (idx < CT) {
#pragma unroll
                for (int j = 0; j < 3; ++j) s_c[b][j][idx] = pc[r][j];
            }
        }
    };

    T Um[3] = {0, 0, 0}, U0[3] = {0, 0, 0}, Wm[3] = {0, 0, 0}, W0[3] = {0, 0, 0};
    T T0[3] = {0, 0, 0}, mc0[3] = {0, 0, 0};
    double err2 = 0.0;
    const int kstart = max(z0 - 1, 0), kend = z1;         // kend may be n3 (no such plane: zeros)
    int cur = 0;
    fetch(kstart);
    stash(0);
    __syncthreads();
    const int lm = (threadIdx.y + 1) * MP + threadIdx.x + 1;
    const int lc = threadIdx.y * CPT + threadIdx.x;        // cell (i1-1, i2-1) of the tile
    for (int k = kstart; k <= kend; ++k) {
        if (k < kend) fetch(k + 1);
        T Up[3], Wp[3], Tn[3], mcn[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const T *t = s_m[cur][j] + lm;
            T P[3], Q[3];
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const T *row = t + (r - 1) * MP;
                const T l = row[-1], c = row[0], rr = row[1];
                Q[r] = eL * (c - l) + eR * (c - rr);
                P[r] = bx0 * c + bxL * l + bxR * rr;
            }
            mcn[j] = t[0];
            const T AyP = fL * (P[1] - P[0]) + fR * (P[1] - P[2]);
            const T ByQ = by0 * Q[1] + byL * Q[0] + byR * Q[2];
            Wp[j] = by0 * P[1] + byL * P[0] + byR * P[2];
            Up[j] = a.idx2[0] * ByQ + a.idx2[1] * AyP;
            const T *cc = s_c[cur][j] + lc;
            Tn[j] = (cc[0] + cc[1]) + (cc[CPT] + cc[CPT + 1]);
        }
        const int z = k - 1;
        if (live && z >= z0 && z < z1) {
            const T gL = z > 0 ? (T)1 : (T)0, gR = z < g.N3 ? (T)1 : (T)0;
            const long long n = (long long)z * pl + (long long)i2 * g.n1 + i1;
            const T sms = UNI_MS ? a.ms_uni * cxy * (gL + gR) : a.sMs[n];
            T H[3] = {0, 0, 0};
            if (sms > 0) {
                const T inv = (T)1 / sms;
                const T bz0 = (gL + gR) * third, bzL = gL * sixth, bzR = gR * sixth;
                T BW[3], an = 0;
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    BW[j] = bz0 * W0[j] + bzL * Wm[j] + bzR * Wp[j];
                    an += a.kax[j] * BW[j];
                }
                const T dsc = UNI_MS ? a.ms_uni * inv : inv;       // demag average weight
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    const T E = (bz0 * U0[j] + bzL * Um[j] + bzR * Up[j]) +
                                a.idx2[2] * (gL * (W0[j] - Wm[j]) + gR * (W0[j] - Wp[j]));
                    T hv = (a.cku * an * a.kax[j] - a.cex * E) * inv + (T0[j] + Tn[j]) * dsc;
                    if (a.terms & NM_TERM_ZEEMAN) hv += a.hu[j];
                    if (a.hadd) hv += a.hadd[j * nn + n];
                    H[j] = hv;
                }
            }
            node_epilogue<T>(a, n, nn, mc0, H, sms, err2);
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            Um[j] = U0[j]; U0[j] = Up[j];
            Wm[j] = W0[j]; W0[j] = Wp[j];
            T0[j] = Tn[j]; mc0[j] = mcn[j];
        }
        if (k < kend) {
            stash(cur ^ 1);
            __syncthreads();
            cur ^= 1;
        }
    }
    if (a.mode == NM_MODE_RK && a.rk.want_err) {
        const double s = block_sum(err2);
        if (tid == 0) a.rk.partials[(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = s;
    }
}

// partials[0..n) -> partials[slot] = sqrt(sum / count), fixed summation order.  `slot` is the fixed last
// entry of the array (its capacity), not n: the commit kernel and the host read-back of a replayed step
// must not depend on which node kernel ran last.
__global__ void k_err_final(double *partials, int n, double count, int slot)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += partials[i];
    const double s = block_sum(v);
    if (threadIdx.x == 0) partials[slot] = sqrt(s / count);
}

// Uniform-field gradient, first pass: per-block fp64 sums of b_n over the nodes with (S Ms)_n > 0.
template <typename T>
__global__ void __launch_bounds__(256) k_hext_partial(const T *__restrict__ m, const T *__restrict__ av,
                                                      const T *__restrict__ sMs, long long nn, T gp, T agp,
                                                      double *__restrict__ part)
{
    double s[3] = {0.0, 0.0, 0.0};
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < nn; n += (long long)gridDim.x * blockDim.x) {
        if (!(sMs[n] > 0)) continue;
        const T mc[3] = {m[n], m[nn + n], m[2 * nn + n]};
        const T ac[3] = {av[n], av[nn + n], av[2 * nn + n]};
        T mxa[3], mxmxa[3];
        cross3(mc, ac, mxa);
        cross3(mc, mxa, mxmxa);
#pragma unroll
        for (int j = 0; j < 3; ++j) s[j] += (double)(gp * mxa[j] - agp * mxmxa[j]);
    }
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double r = block_sum(s[j]);
        if (threadIdx.x == 0) part[j * gridDim.x + blockIdx.x] = r;
        __syncthreads();                                    // block_sum's scratch is reused
    }
}

// second pass: u_h[j] += coef * (-sum of the block sums), fixed order
__global__ void k_hext_final(const double *__restrict__ part, int nblocks, double coef, double *__restrict__ u_h)
{
    for (int j = 0; j < 3; ++j) {
        double v = 0.0;
        for (int i = threadIdx.x; i < nblocks; i += blockDim.x) v += part[j * nblocks + i];
        const double r = block_sum(v);
        if (threadIdx.x == 0) u_h[j] += coef * (-r);
        __syncthreads();
    }
}

// VJPs with respect to the cell-wise A and Ku: one thread per cell gathers m, a and S Ms of its 8 vertices.
template <typename T> __global__ void __launch_bounds__(128) k_mat_grad(const NmMatGradArgs<T> a)
{
    const NmGeom &g = a.g;
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= g.cells) return;
    const int c1 = (int)(c % g.N1), c2 = (int)((c / g.N1) % g.N2), c3 = (int)(c / ((long long)g.N1 * g.N2));
    const long long nn = g.nodes;
    T mv[8][3], bl[8][3], mk[8], bk[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        // strides g.ys / g.zs: 0 along a reduced axis (the two vertices are one node; a.invL carries the 2^D / 8)
        const long long n = (long long)(c3 + ((i >> 2) & 1)) * g.zs + (long long)(c2 + ((i >> 1) & 1)) * g.ys + (c1 + (i & 1));
        const T mc[3] = {a.m[n], a.m[nn + n], a.m[2 * nn + n]};
        const T ac[3] = {a.a[n], a.a[nn + n], a.a[2 * nn + n]};
        const T sms = a.sMs[n];
        const T il = sms > 0 ? a.invL / sms : (T)0;
        T mxa[3], mxmxa[3];
        cross3(mc, ac, mxa);
        cross3(mc, mxa, mxmxa);
        mk[i] = 0;
        bk[i] = 0;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            mv[i][j] = mc[j];
            bl[i][j] = (a.gp * mxa[j] - a.agp * mxmxa[j]) * il;
            mk[i] += mc[j] * a.kax[j];
            bk[i] += bl[i][j] * a.kax[j];
        }
    }
    T gA = 0, gKu = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int ip = 0; ip < 8; ++ip) {
            const int e = i ^ ip;
            gA += a.wK[e] * (bl[i][0] * mv[ip][0] + bl[i][1] * mv[ip][1] + bl[i][2] * mv[ip][2]);
            gKu += a.wM[e] * bk[i] * mk[ip];
        }
    gA = a.ex_on ? (T)2 * gA : (T)0;
    gKu = a.an_on ? (T)-2 * gKu : (T)0;
    if (a.u_A) a.u_A[c] = a.accumulate ? a.u_A[c] + a.coef * gA : gA;
    if (a.u_Ku) a.u_Ku[c] = a.accumulate ? a.u_Ku[c] + a.coef * gKu : gKu;
}

// Dormand-Prince commit: m <- (normalised) y5 iff err <= 1
template <typename T>
__global__ void k_commit(T *__restrict__ m, const T *__restrict__ y5, long long nodes,
                         const double *__restrict__ err, int renorm)
{
    if (!(*err <= 1.0)) return;
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= nodes) return;
    T y[3] = {y5[n], y5[nodes + n], y5[2 * nodes + n]};
    if (renorm) {
        const T n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
        const T inv = n2 > (T)0 ? rsqrt_t<T>(n2) : (T)0;   // a zero vector (vacuum node) stays zero
        y[0] *= inv; y[1] *= inv; y[2] *= inv;
    }
    m[n] = y[0]; m[nodes + n] = y[1]; m[2 * nodes + n] = y[2];
}

template <typename T>
__global__ void k_sMs(const T *__restrict__ Ms, T *__restrict__ sMs, NmGeom g)
{
    const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= g.nodes) return;
    const int i1 = (int)(n % g.n1), i2 = (int)((n / g.n1) % g.n2), i3 = (int)(n / ((long long)g.n1 * g.n2));
    T s = 0;
    for (int oz = 0; oz < 2; ++oz)
        for (int oy = 0; oy < 2; ++oy)
            for (int ox = 0; ox < 2; ++ox) {
                const int c1 = i1 + ox - 1, c2 = i2 + oy - 1, c3 = i3 + oz - 1;
                if (c1 >= 0 && c1 < g.N1 && c2 >= 0 && c2 < g.N2 && c3 >= 0 && c3 < g.N3)
                    s += Ms[((long long)c3 * g.N2 + c2) * g.N1 + c1];
            }
    sMs[n] = s;
}

// a11, Ms gradient per cell (reading C7):
//   dudt_c = -[ -(S^T w)_c + zeeman piece + (S^T q)_c . Hcell_c + mbar_c . Y_c ],  Y = 8 Hc2
template <typename T>
__global__ void k_adj_cell(const NmAdjCellArgs<T> a)
{
    const NmGeom &g = a.g;
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= g.cells) return;
    const int c1 = (int)(c % g.N1), c2 = (int)((c / g.N1) % g.N2), c3 = (int)(c / ((long long)g.N1 * g.N2));
    const long long nn = g.nodes;
    T sw = 0, sq[3] = {0, 0, 0}, sm[3] = {0, 0, 0}, zee = 0;
    const bool zee_on = (a.terms & NM_TERM_ZEEMAN) != 0;
    const bool zee_nodal = zee_on && (a.h_static || a.h_pulse);
    long long nd[8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
        nd[i] = (long long)(c3 + (i >> 2)) * g.zs + (long long)(c2 + ((i >> 1) & 1)) * g.ys + (c1 + (i & 1));
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        sw += a.W[nd[i]];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            sq[j] += a.Q[j * nn + nd[i]];
            sm[j] += a.m[j * nn + nd[i]];
        }
    }
    if (zee_nodal) {
        for (int ip = 0; ip < 8; ++ip) {
            T h[3];
            for (int j = 0; j < 3; ++j) {
                T v = 0;
                if (a.h_static) v += a.h_static[j * nn + nd[ip]];
                if (a.h_pulse) v += a.amp * a.h_pulse[j * nn + nd[ip]];
                h[j] = v;
            }
            for (int i = 0; i < 8; ++i) {
                const T w = a.wM8V[i ^ ip];
                zee += w * (a.Q[nd[i]] * h[0] + a.Q[nn + nd[i]] * h[1] + a.Q[2 * nn + nd[i]] * h[2]);
            }
        }
    }
    if (zee_on) zee += sq[0] * a.hu[0] + sq[1] * a.hu[1] + sq[2] * a.hu[2];
    T grad = -sw + zee;
    if (a.Hc1) {
        for (int j = 0; j < 3; ++j)
            grad += sq[j] * a.Hc1[j * g.cells + c] + sm[j] * a.Hc2[j * g.cells + c];   // mbar.Y = (sm/8).(8 Hc2)
    }
    // reduced basis (strides 0): every vertex of the 2^D was counted 2^(3-D) times in each of the four pieces
    a.dudt[c] = -grad * a.red;
}

// The same without nodal Zeeman arrays, marching along z: a thread owns one cell column (c1, c2) of
// a z chunk and keeps the sums over the four nodes (c1 + {0,1}, c2 + {0,1}) of the previous node
// plane, so every plane costs four loads per array instead of eight (rows of a warp are contiguous;
// the x + 1 / y + 1 overlaps are served by L1).
template <typename T>
__global__ void __launch_bounds__(256) k_adj_cell_march(const NmAdjCellArgs<T> a, int zchunk)
{
    const NmGeom &g = a.g;
    const int c1 = blockIdx.x * 32 + threadIdx.x, c2 = blockIdx.y * 8 + threadIdx.y;
    if (c1 >= g.N1 || c2 >= g.N2) return;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, g.N3);
    const long long nn = g.nodes;
    const long long pl = (long long)g.n1 * g.n2;
    const bool zee_on = (a.terms & NM_TERM_ZEEMAN) != 0;
    T pw = 0, pq[3] = {0, 0, 0}, pm[3] = {0, 0, 0};
    const T *w0 = a.W + (long long)z0 * pl + (long long)c2 * g.n1 + c1;
    const T *q0 = a.Q + (long long)z0 * pl + (long long)c2 * g.n1 + c1;
    const T *m0 = a.m + (long long)z0 * pl + (long long)c2 * g.n1 + c1;
    long long c = ((long long)z0 * g.N2 + c2) * g.N1 + c1;
    const long long cpl = (long long)g.N1 * g.N2;
    for (int k = z0; k <= z1; ++k, w0 += pl, q0 += pl, m0 += pl) {
        const int r1 = g.n1;
        const T cw = (w0[0] + w0[1]) + (w0[r1] + w0[r1 + 1]);
        T cq[3], cm[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const T *q = q0 + j * nn, *m = m0 + j * nn;
            cq[j] = (q[0] + q[1]) + (q[r1] + q[r1 + 1]);
            cm[j] = (m[0] + m[1]) + (m[r1] + m[r1 + 1]);
        }
        if (k > z0) {          // cell plane k - 1
            const T sw = pw + cw;
            T grad = -sw;
            T sq[3], sm[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                sq[j] = pq[j] + cq[j];
                sm[j] = pm[j] + cm[j];
            }
            if (zee_on) grad += sq[0] * a.hu[0] + sq[1] * a.hu[1] + sq[2] * a.hu[2];
            if (a.Hc1) {
#pragma unroll
                for (int j = 0; j < 3; ++j) grad += sq[j] * a.Hc1[j * g.cells + c] + sm[j] * a.Hc2[j * g.cells + c];
            }
            a.dudt[c] = -grad;
            c += cpl;
        }
        pw = cw;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            pq[j] = cq[j];
            pm[j] = cm[j];
        }
    }
}

// out = base + sum_j coef_j src_j  (optionally normalised as 3-vectors over `vec_n` nodes)
template <typename T> struct LinArgs {
    T *out;
    const T *base;
    const T *src[4];
    T coef[4];
    int nsrc;
    long long n;        // elements
    long long vec_n;    // > 0: arrays are [3][vec_n] and the result is normalised per node
};

template <typename T> __global__ void k_lincomb(const LinArgs<T> a)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a.vec_n > 0) {
        if (i >= a.vec_n) return;
        T y[3];
        for (int j = 0; j < 3; ++j) {
            T v = a.base[j * a.vec_n + i];
            for (int s = 0; s < a.nsrc; ++s) v += a.coef[s] * a.src[s][j * a.vec_n + i];
            y[j] = v;
        }
        const T n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
        const T inv = n2 > (T)0 ? rsqrt_t<T>(n2) : (T)0;   // a zero vector (vacuum node) stays zero
        for (int j = 0; j < 3; ++j) a.out[j * a.vec_n + i] = y[j] * inv;
    } else {
        if (i >= a.n) return;
        T v = a.base[i];
        for (int s = 0; s < a.nsrc; ++s) v += a.coef[s] * a.src[s][i];
        a.out[i] = v;
    }
}

// Up to NM_LIN_OPS independent out = base + coef src updates in one launch (blockIdx.y = update):
// the stage updates of the adjoint Runge-Kutta step.  Same arithmetic as k_lincomb with one source.
template <typename T> struct LinBatch {
    LinArgs<T> op[NM_LIN_OPS];
};

template <typename T> __global__ void k_lincomb_batch(const LinBatch<T> b)
{
    const LinArgs<T> &a = b.op[blockIdx.y];
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a.vec_n > 0) {
        if (i >= a.vec_n) return;
        T y[3];
        for (int j = 0; j < 3; ++j) {
            T v = a.base[j * a.vec_n + i];
            v += a.coef[0] * a.src[0][j * a.vec_n + i];
            y[j] = v;
        }
        const T n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
        const T inv = n2 > (T)0 ? rsqrt_t<T>(n2) : (T)0;   // a zero vector (vacuum node) stays zero
        for (int j = 0; j < 3; ++j) a.out[j * a.vec_n + i] = y[j] * inv;
    } else {
        if (i >= a.n) return;
        T v = a.base[i];
        v += a.coef[0] * a.src[0][i];
        a.out[i] = v;
    }
}

inline unsigned nblk(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// Grid of k_node_sep: SX x SY patches of node columns, z split into chunks so that about eight
// CTAs per SM exist (each chunk re-reads one halo plane on either side).
inline dim3 sep_grid(const NmGeom &g, int *zchunk)
{
    const unsigned gx = nblk(g.n1, SX), gy = nblk(g.n2, SY);
    int gz = (int)((148 * 8 + gx * gy - 1) / (gx * gy));
    const int gz_max = g.n3 / 8 > 1 ? g.n3 / 8 : 1;
    if (gz > gz_max) gz = gz_max;
    if (gz < 1) gz = 1;
    *zchunk = (g.n3 + gz - 1) / gz;
    return dim3(gx, gy, nblk(g.n3, *zchunk));
}


// -------------------------------------------------------------------------------------------------
// Further local terms through the weak form (readings F3), one thread per
// node, the paper's element loop (Eqs. 19-20) gathered: for each of the (up to 8) cells c that contain
// node n = c + i,
//   DMI     dE_{n,a} += D_c sum_{d,b} T[a,d,b] g_d[b],   g_d = sum_{i'} (G^d[i,i'] - G^d[i',i]) m_{c+i'}
//           with G^d[i,i'] - G^d[i',i] = (V / dx_d) (i'_d - i_d) M1[i_e,i'_e] M1[i_f,i'_f]  (M1 = 1/3, 1/6):
//           T antisymmetric in (a, b): the Levi-Civita symbol (bulk) or T[n,d,d] = 1, T[d,d,n] = -1 (interfacial)
//   cubic   dE_{n,j} += Kc_c V sum_q w_q phi_i(x_q) de/dm_j(m^h(x_q)),  3-point Gauss rule per axis (exact),
//           e = a1^2 a2^2 + a2^2 a3^2 + a3^2 a1^2,  a_r = m . c_r,  de/dm = sum_r 2 a_r (|a|^2 - a_r^2) c_r
//           (adjoint pass 2: the Hessian of that energy at m applied to q instead, which is what (dH_cub/dm)^T b is)
// out_n = -dE_n / L_n, L_n = mu0 (V/8) (S Ms)_n (Eq. 22); 0 where (S Ms)_n = 0.
template <typename T>
__global__ void __launch_bounds__(kBlock) k_extra_local(const NmExtraArgs<T> a)
{
    const NmGeom &g = a.g;
    const int pl = g.n1 * g.n2;
    const int p = blockIdx.x * kBlock + threadIdx.x;
    const int i3 = blockIdx.y;
    if (p >= pl) return;
    const int i2 = p / g.n1, i1 = p - i2 * g.n1;
    const long long nn = g.nodes;
    const long long n = (long long)i3 * pl + p;
    const T third = (T)(1.0 / 3.0), sixth = (T)(1.0 / 6.0);
    // 3-point Gauss-Legendre rule on [0, 1]
    const T gx[3] = {(T)(0.5 - 0.5 * 0.77459666924148337704), (T)0.5, (T)(0.5 + 0.5 * 0.77459666924148337704)};
    const T gw[3] = {(T)(5.0 / 18.0), (T)(8.0 / 18.0), (T)(5.0 / 18.0)};
    T dE[3] = {0, 0, 0};
    T sms = 0;
    for (int ci = 0; ci < 8; ++ci) {
        const int bx = ci & 1, by = (ci >> 1) & 1, bz = ci >> 2;     // 0: the cell below the node along that axis
        const int c1 = i1 - 1 + bx, c2 = i2 - 1 + by, c3 = i3 - 1 + bz;
        if (c1 < 0 || c1 >= g.N1 || c2 < 0 || c2 >= g.N2 || c3 < 0 || c3 >= g.N3) continue;
        const long long c = ((long long)c3 * g.N2 + c2) * g.N1 + c1;
        sms += a.Ms[c];
        const int iv[3] = {1 - bx, 1 - by, 1 - bz};                  // local vertex index of n in cell c
        const long long n0 = ((long long)c3 * g.n2 + c2) * g.n1 + c1; // vertex (0,0,0) of the cell
        T mv[8][3];
#pragma unroll
        for (int v = 0; v < 8; ++v) {
            const long long q = n0 + (v & 1) + ((v >> 1) & 1) * g.n1 + (long long)(v >> 2) * pl;
            mv[v][0] = a.fld[q];
            mv[v][1] = a.fld[nn + q];
            mv[v][2] = a.fld[2 * nn + q];
        }
        if (a.D) {
            T gd[3][3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                gd[d][0] = gd[d][1] = gd[d][2] = 0;
#pragma unroll
                for (int v = 0; v < 8; ++v) {
                    const int vv[3] = {v & 1, (v >> 1) & 1, v >> 2};
                    const int sd = vv[d] - iv[d];
                    if (sd == 0) continue;
                    T w = (T)sd * a.V * a.idx[d];
#pragma unroll
                    for (int e = 0; e < 3; ++e)
                        if (e != d) w *= (vv[e] == iv[e]) ? third : sixth;
                    gd[d][0] += w * mv[v][0];
                    gd[d][1] += w * mv[v][1];
                    gd[d][2] += w * mv[v][2];
                }
            }
            const T Dc = a.D[c];
            if (a.dmi_kind == 0) {      // sum_{d,b} eps[a,d,b] g_d[b]
                dE[0] += Dc * (gd[1][2] - gd[2][1]);
                dE[1] += Dc * (gd[2][0] - gd[0][2]);
                dE[2] += Dc * (gd[0][1] - gd[1][0]);
            } else {
                const int nrm = a.dmi_normal;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    if (d == nrm) continue;
                    dE[nrm] += Dc * gd[d][d];       // T[n,d,d] = +1
                    dE[d] -= Dc * gd[d][nrm];       // T[d,d,n] = -1
                }
            }
        }
        if (a.Kc) {
            const T KV = a.Kc[c] * a.V;
            // a.about != null: the Hessian of the energy at `about` applied to fld (adjoint pass 2) instead of the
            // gradient at fld:  d2e/da_r da_s = 2 (|a|^2 - a_r^2) delta_rs + 4 a_r a_s (1 - delta_rs)
            T av[8][3];
            if (a.about) {
#pragma unroll
                for (int v = 0; v < 8; ++v) {
                    const long long q = n0 + (v & 1) + ((v >> 1) & 1) * g.n1 + (long long)(v >> 2) * pl;
                    av[v][0] = a.about[q];
                    av[v][1] = a.about[nn + q];
                    av[v][2] = a.about[2 * nn + q];
                }
            }
            for (int qz = 0; qz < 3; ++qz)
                for (int qy = 0; qy < 3; ++qy)
#pragma unroll
                    for (int qx = 0; qx < 3; ++qx) {
                        const T fx[2] = {(T)1 - gx[qx], gx[qx]}, fy[2] = {(T)1 - gx[qy], gx[qy]}, fz[2] = {(T)1 - gx[qz], gx[qz]};
                        T mq[3] = {0, 0, 0}, aq[3] = {0, 0, 0};
#pragma unroll
                        for (int v = 0; v < 8; ++v) {
                            const T ph = fx[v & 1] * fy[(v >> 1) & 1] * fz[v >> 2];
                            mq[0] += ph * mv[v][0];
                            mq[1] += ph * mv[v][1];
                            mq[2] += ph * mv[v][2];
                            if (a.about) {
                                aq[0] += ph * av[v][0];
                                aq[1] += ph * av[v][1];
                                aq[2] += ph * av[v][2];
                            }
                        }
                        const T wq = KV * gw[qx] * gw[qy] * gw[qz] * fx[iv[0]] * fy[iv[1]] * fz[iv[2]];
                        if (!a.about) {
                            T al[3], S = 0;
#pragma unroll
                            for (int r = 0; r < 3; ++r) {
                                al[r] = a.cax[3 * r] * mq[0] + a.cax[3 * r + 1] * mq[1] + a.cax[3 * r + 2] * mq[2];
                                S += al[r] * al[r];
                            }
#pragma unroll
                            for (int r = 0; r < 3; ++r) {
                                const T cr = (T)2 * al[r] * (S - al[r] * al[r]) * wq;
                                dE[0] += cr * a.cax[3 * r];
                                dE[1] += cr * a.cax[3 * r + 1];
                                dE[2] += cr * a.cax[3 * r + 2];
                            }
                        } else {
                            T al[3], be[3], S = 0, ab = 0;
#pragma unroll
                            for (int r = 0; r < 3; ++r) {
                                al[r] = a.cax[3 * r] * aq[0] + a.cax[3 * r + 1] * aq[1] + a.cax[3 * r + 2] * aq[2];
                                be[r] = a.cax[3 * r] * mq[0] + a.cax[3 * r + 1] * mq[1] + a.cax[3 * r + 2] * mq[2];
                                S += al[r] * al[r];
                                ab += al[r] * be[r];
                            }
#pragma unroll
                            for (int r = 0; r < 3; ++r) {
                                const T cr = ((T)2 * (S - al[r] * al[r]) * be[r] + (T)4 * al[r] * (ab - al[r] * be[r])) * wq;
                                dE[0] += cr * a.cax[3 * r];
                                dE[1] += cr * a.cax[3 * r + 1];
                                dE[2] += cr * a.cax[3 * r + 2];
                            }
                        }
                    }
        }
    }
    // interlayer coupling: dE_{(f+i, z_a)} += -J dx dy sum_{i'} M1 M1 m_{(f+i', z_b)} over the (up to 4) faces f of the
    // node in its plane, and the same with the planes exchanged
    if (a.rkky_JA != (T)0 && (i3 == a.rkky_za || i3 == a.rkky_zb)) {
        const int zo = i3 == a.rkky_za ? a.rkky_zb : a.rkky_za;
        for (int fi = 0; fi < 4; ++fi) {
            const int bx = fi & 1, by = fi >> 1;
            const int f1 = i1 - 1 + bx, f2 = i2 - 1 + by;
            if (f1 < 0 || f1 >= g.N1 || f2 < 0 || f2 >= g.N2) continue;
            const int ix = 1 - bx, iy = 1 - by;                      // local vertex of the node in face f
#pragma unroll
            for (int v = 0; v < 4; ++v) {
                const int vx = v & 1, vy = v >> 1;
                const T w = -a.rkky_JA * (vx == ix ? third : sixth) * (vy == iy ? third : sixth);
                const long long q = (long long)zo * pl + (long long)(f2 + vy) * g.n1 + (f1 + vx);
                dE[0] += w * a.fld[q];
                dE[1] += w * a.fld[nn + q];
                dE[2] += w * a.fld[2 * nn + q];
            }
        }
    }
    const T sc = sms > 0 ? (T)-1 / (a.mu0V8 * sms) : (T)0;
#pragma unroll
    for (int j = 0; j < 3; ++j) a.out[j * nn + n] = sc * dE[j];
}

} // namespace

// ---- host launchers used by nm_api.cu -----------------------------------------------------------
template <typename T> nm_status nm_launch_node(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    const bool nodal_zee = (a.terms & NM_TERM_ZEEMAN) && (a.h_static || a.h_pulse);
    const bool fwd_mode = a.mode == NM_MODE_H || a.mode == NM_MODE_RHS || a.mode == NM_MODE_RK;
    if (a.sep && nodal_zee && fwd_mode && mesh->Zs) {
        // nodal Zeeman arrays with uniform A and Ku: smooth the field once, then the separable kernels
        {
            NmLaunchScope sc(mesh, NM_K_OTHER, st);
            const dim3 grid((a.g.n1 + ZX - 1) / ZX, (a.g.n2 + ZY - 1) / ZY, a.g.n3);
            k_zeeman_smooth<T, false><<<grid, dim3(ZX, ZY), 0, st>>>(a, (T *)mesh->Zs, (T)0, 0);
        }
        NM_CUDA_TRY(cudaGetLastError());
        NmLocalArgs<T> b = a;
        b.h_static = b.h_pulse = nullptr;
        b.hadd = (const T *)mesh->Zs;
        return nm_launch_node<T>(mesh, b, st);
    }
    if (a.sep == 1 && !nodal_zee && nm_node_col_ok<T>(mesh, a)) return nm_launch_node_col<T>(mesh, a, st);
    if (a.sep && !nodal_zee) {
        int zchunk;
        const dim3 grid = sep_grid(a.g, &zchunk);
        mesh->last_partials = (int)(grid.x * grid.y * grid.z);
        NmLaunchScope sc(mesh, nm_node_class(a.mode), st);
        if (a.ms_uni > 0) k_node_sep<T, true><<<grid, dim3(SX, SY), 0, st>>>(a, zchunk);
        else k_node_sep<T, false><<<grid, dim3(SX, SY), 0, st>>>(a, zchunk);
    } else {
        NmLaunchScope sc(mesh, nm_node_class(a.mode), st);
        const dim3 grid(nblk((long long)a.g.n1 * a.g.n2, kBlock), a.g.n3);
        mesh->last_partials = (int)(grid.x * grid.y);
        const bool extra = (a.terms & NM_TERM_ANISO) || nodal_zee;
        if (extra) k_node<T, true><<<grid, kBlock, 0, st>>>(a);
        else k_node<T, false><<<grid, kBlock, 0, st>>>(a);
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T> nm_status nm_launch_extra(nm_mesh *mesh, const NmExtraArgs<T> &a, cudaStream_t st)
{
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        const dim3 grid(nblk((long long)a.g.n1 * a.g.n2, kBlock), a.g.n3);
        k_extra_local<T><<<grid, kBlock, 0, st>>>(a);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}
template nm_status nm_launch_extra<float>(nm_mesh *, const NmExtraArgs<float> &, cudaStream_t);
template nm_status nm_launch_extra<double>(nm_mesh *, const NmExtraArgs<double> &, cudaStream_t);

int nm_node_blocks(const NmGeom &g)
{
    int zchunk;
    const dim3 sg = sep_grid(g, &zchunk);
    const int gen = (int)(nblk((long long)g.n1 * g.n2, kBlock) * g.n3);
    const int sep = (int)(sg.x * sg.y * sg.z);
    const int col = nm_node_col_blocks(g);
    return gen > sep ? (gen > col ? gen : col) : (sep > col ? sep : col);
}

nm_status nm_launch_err_final(nm_mesh *mesh, int n_partials, double count, cudaStream_t st)
{
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        k_err_final<<<1, 1024, 0, st>>>(mesh->partials, n_partials, count, mesh->n_partials);
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T> nm_status nm_launch_mat_grad(nm_mesh *mesh, const NmMatGradArgs<T> &a, cudaStream_t st)
{
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        k_mat_grad<T><<<nblk(a.g.cells, 128), 128, 0, st>>>(a);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T>
nm_status nm_launch_hext_grad(nm_mesh *mesh, const T *m, const T *a, double gp, double agp, double coef,
                              double *u_h, cudaStream_t st)
{
    const long long nn = mesh->g.nodes;
    long long nb = (nn + 255) / 256;
    if (nb > NM_HEXT_BLOCKS) nb = NM_HEXT_BLOCKS;
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        k_hext_partial<T><<<(unsigned)nb, 256, 0, st>>>(m, a, (const T *)mesh->sMs, nn, (T)gp, (T)agp, mesh->hpart);
    }
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        k_hext_final<<<1, 256, 0, st>>>(mesh->hpart, (int)nb, coef, u_h);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

// u_hn (+)= coef Z(q L / L) with q = b / (S Ms) given (q != null: the Q array of the adjoint pass) or made here
// from (m, a) into the mesh's Q scratch
template <typename T>
nm_status nm_launch_hnodal_grad(nm_mesh *mesh, const NmLocalArgs<T> &base, const T *q, const T *m, const T *av,
                                double coef, int accumulate, T *u_hn, cudaStream_t st)
{
    const long long nn = mesh->g.nodes;
    if (!q) {
        {
            NmLaunchScope sc(mesh, NM_K_OTHER, st);
            k_bq<T><<<nblk(nn, 256), 256, 0, st>>>(m, av, (const T *)mesh->sMs, nn, base.gp, base.agp, (T *)mesh->Q);
        }
        q = (const T *)mesh->Q;
    }
    NmLocalArgs<T> a = base;
    a.h_static = q;
    a.h_pulse = nullptr;
    a.hadd = nullptr;
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        const dim3 grid((a.g.n1 + ZX - 1) / ZX, (a.g.n2 + ZY - 1) / ZY, a.g.n3);
        k_zeeman_smooth<T, true><<<grid, dim3(ZX, ZY), 0, st>>>(a, u_hn, (T)coef, accumulate);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T>
nm_status nm_launch_commit(nm_mesh *mesh, T *m, const T *y5, const double *err, int renorm, cudaStream_t st)
{
    {
        NmLaunchScope sc(mesh, NM_K_OTHER, st);
        k_commit<T><<<nblk(mesh->g.nodes, 256), 256, 0, st>>>(m, y5, mesh->g.nodes, err, renorm);
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T> nm_status nm_launch_adj_cell(nm_mesh *mesh, const NmAdjCellArgs<T> &a, cudaStream_t st)
{
    {
        NmLaunchScope sc(mesh, NM_K_ADJ_CELL, st);
        const bool zee_nodal = (a.terms & NM_TERM_ZEEMAN) && (a.h_static || a.h_pulse);
        if (zee_nodal || a.g.N3 < 32) k_adj_cell<T><<<nblk(a.g.cells, 128), 128, 0, st>>>(a);
        else {
            // z chunks of 4..32 planes, short enough for about eight CTAs per SM
            const int base = ((a.g.N1 + 31) / 32) * ((a.g.N2 + 7) / 8);
            const int nz = (8 * mesh->sm_count + base - 1) / base;
            int zchunk = (a.g.N3 + nz - 1) / nz;
            zchunk = zchunk < 4 ? 4 : (zchunk > 32 ? 32 : zchunk);
            const dim3 grid((a.g.N1 + 31) / 32, (a.g.N2 + 7) / 8, (a.g.N3 + zchunk - 1) / zchunk);
            k_adj_cell_march<T><<<grid, dim3(32, 8), 0, st>>>(a, zchunk);
        }
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T>
nm_status nm_lincomb(nm_mesh *mesh, T *out, const T *base, int nsrc, const T *const *src, const T *coef,
                     long long n, long long vec_n, cudaStream_t st)
{
    LinArgs<T> a;
    a.out = out; a.base = base; a.nsrc = nsrc; a.n = n; a.vec_n = vec_n;
    for (int s = 0; s < 4; ++s) {
        a.src[s] = s < nsrc ? src[s] : nullptr;
        a.coef[s] = s < nsrc ? coef[s] : (T)0;
    }
    {
        NmLaunchScope sc(mesh, NM_K_LINCOMB, st);
        k_lincomb<T><<<nblk(vec_n > 0 ? vec_n : n, 256), 256, 0, st>>>(a);
    }

    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T>
nm_status nm_lincomb_batch(nm_mesh *mesh, const NmLinOp<T> *ops, int nops, cudaStream_t st)
{
    if (nops < 1 || nops > NM_LIN_OPS) { nm_set_error("nm_lincomb_batch: %d updates", nops); return NM_EINVAL; }
    LinBatch<T> b;
    memset(&b, 0, sizeof(b));
    long long longest = 0;
    for (int o = 0; o < nops; ++o) {
        LinArgs<T> &a = b.op[o];
        a.out = ops[o].out; a.base = ops[o].base; a.nsrc = 1; a.n = ops[o].n; a.vec_n = ops[o].vec_n;
        a.src[0] = ops[o].src;
        a.coef[0] = ops[o].coef;
        const long long threads = a.vec_n > 0 ? a.vec_n : a.n;
        if (threads > longest) longest = threads;
    }
    {
        NmLaunchScope sc(mesh, NM_K_LINCOMB, st);
        k_lincomb_batch<T><<<dim3(nblk(longest, 256), nops), 256, 0, st>>>(b);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

nm_status nm_compute_sMs(nm_mesh *mesh, cudaStream_t st)
{
    NmLaunchScope sc(mesh, NM_K_OTHER, st);
    if (mesh->f64)
        k_sMs<double><<<nblk(mesh->g.nodes, 256), 256, 0, st>>>((const double *)mesh->Ms, (double *)mesh->sMs, mesh->g);
    else
        k_sMs<float><<<nblk(mesh->g.nodes, 256), 256, 0, st>>>((const float *)mesh->Ms, (float *)mesh->sMs, mesh->g);
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

#define NM_INST(T)                                                                                       \
    template nm_status nm_launch_node<T>(nm_mesh *, const NmLocalArgs<T> &, cudaStream_t);              \
    template nm_status nm_launch_commit<T>(nm_mesh *, T *, const T *, const double *, int, cudaStream_t); \
    template nm_status nm_launch_mat_grad<T>(nm_mesh *, const NmMatGradArgs<T> &, cudaStream_t);        \
    template nm_status nm_launch_hext_grad<T>(nm_mesh *, const T *, const T *, double, double, double,  \
                                              double *, cudaStream_t);                                  \
    template nm_status nm_launch_adj_cell<T>(nm_mesh *, const NmAdjCellArgs<T> &, cudaStream_t);        \
    template nm_status nm_launch_hnodal_grad<T>(nm_mesh *, const NmLocalArgs<T> &, const T *, const T *, const T *, \
                                                double, int, T *, cudaStream_t);                       \
    template nm_status nm_lincomb<T>(nm_mesh *, T *, const T *, int, const T *const *, const T *,       \
                                     long long, long long, cudaStream_t);                               \
    template nm_status nm_lincomb_batch<T>(nm_mesh *, const NmLinOp<T> *, int, cudaStream_t);
NM_INST(float)
NM_INST(double)
