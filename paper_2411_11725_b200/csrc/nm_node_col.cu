// Column-marching node kernel: a5-a11 of the hot path for uniform A and Ku.
//
// The assembled tensor-product element operators of Eqs. (17)-(22) (reading C2) factor into 1-D
// stiffness and mass operators along each axis,
//     (A v)_i = [i>0] (v_i - v_{i-1}) + [i<N] (v_i - v_{i+1}),
//     (B v)_i = [i>0] (v_i/3 + v_{i-1}/6) + [i<N] (v_i/3 + v_{i+1}/6)   =   d_i v_i - (A v)_i / 6,
// with d_i = 1 inside and 1/2 on the two end nodes (the 1-D lumped mass), and A is the plain
// interior formula 2 v_i - v_{i-1} - v_{i+1} on data whose ghost nodes mirror the end nodes.  So
//     E_n   = dx^-2 (Bz By Ax m) + dy^-2 (Bz Ay Bx m) + dz^-2 (Az By Bx m)
//     H^ex  = -(16 A / (mu0 (S Ms)_n)) E_n,   H^an = (16 Ku / (mu0 (S Ms)_n)) (Bz By Bx (m.k)) k
//     H^d_n = S(Ms o H^cell)_n / (S Ms)_n                                     (reading C5)
// needs, per plane, only ax = Ax m, ay = Ay m and axy = Ay Ax m of the 3 x 3 neighbourhood:
//     U = dx^-2 By Ax m + dy^-2 Ay Bx m = dx^-2 dy ax + dy^-2 dx ay - (dx^-2 + dy^-2)/6 axy
//     W = By Bx m                       = dx dy m - dy/6 ax - dx/6 ay + axy/36
//     E_z = dz U_z + (Az R)_z,   R = dz^-2 W - U/6;      (Bz W)_z = dz W_z - (Az W)_z / 6
// (dx, dy, dz here: the factors d of the node along each axis) and no per-neighbour boundary
// coefficients.  The z operators are accumulated plane by plane in two partial sums per output
// (the sum that still waits for plane k + 1, and the start of the next one), so the march carries
// 8 registers per node and no register rotation.  Then the LLG products (Eq. 1), the
// Runge-Kutta stage combination (a10) or the adjoint products (a11, reading C7).
//
// How the SM is fed: a CTA owns RY whole node rows (one thread per node column i1, so every global
// and shared access of a warp is a contiguous row segment) and marches along z.  A plane's tile --
// RY + 2 node rows of each component of m with one ghost column either side, fetched at clamped
// (mirrored) row / column indices; RY + 1 cell rows of each component of H^cell (and of Ms),
// zero-filled outside the mesh -- is streamed by cp.async into a ring of CS stages, CS - 2 planes
// ahead of the arithmetic, one CTA barrier per plane.  The epilogue is compiled per mode.
#include "nm_async.cuh"
#include "nm_local.cuh"
#include "nm_pair.cuh"

using namespace nmp;
using namespace nma;

namespace {

// A pair = the same quantity on the two node rows (ry = 0, 1) a thread owns: fp32 pairs run on the
// packed instructions of nm_pair.cuh, fp64 pairs on scalar ones.
template <typename T> struct PairOf { typedef typename NmVec2<T>::type V; };
template <typename T> __device__ __forceinline__ typename PairOf<T>::V pr(T a, T b)
{
    typename PairOf<T>::V v;
    v.x = a;
    v.y = b;
    return v;
}
template <typename T> __device__ __forceinline__ typename PairOf<T>::V pr1(T a) { return pr<T>(a, a); }
template <typename V> __device__ __forceinline__ V pneg(V a) { a.x = -a.x; a.y = -a.y; return a; }

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

template <typename T> __device__ __forceinline__ T rcp_c(T v);
template <> __device__ __forceinline__ float rcp_c<float>(float v) { return __fdividef(1.0f, v); }
template <> __device__ __forceinline__ double rcp_c<double>(double v) { return 1.0 / v; }

// modes of the compiled epilogues: the NmLocalMode values, with the Runge-Kutta stage split by the
// way it combines (RK0: no earlier derivative, the first stages of RK4; RKS: last stage of RK4 from the
// stage states; RKN: a loop over stored derivatives, Dormand-Prince)
enum { CM_H = 0, CM_RHS, CM_RK0, CM_RKS, CM_RKN, CM_ADJ1, CM_ADJ2, CM_COUNT };

// element n of component j of a nodal vector array (n < nodes < 2^31: one 32-bit index per node)
template <typename P> __device__ __forceinline__ P *comp(P *base, int j, size_t nn) { return base + j * nn; }

// a10-a11 on one node.  mc = fld_n, f = the LLG right-hand side (a9, computed by the caller for both
// rows at once), sms = (S Ms)_n; y0 = what the mode reads at this node, loaded before the plane
// arithmetic: the start-of-step state (Runge-Kutta), a (ADJ1) or d (ADJ2).
template <typename T, int CM>
__device__ __forceinline__ void epilogue_c(const NmLocalArgs<T> &a, unsigned n, size_t nn, const T *mc,
                                           const T *H, const T *f, T sms, const T *y0, const T *sp, double &err2)
{
    if (CM == CM_H) {
#pragma unroll
        for (int j = 0; j < 3; ++j) comp(a.out, j, nn)[n] = H[j];
        return;
    }
    if (CM == CM_ADJ2) {
#pragma unroll
        for (int j = 0; j < 3; ++j) comp(a.dadt, j, nn)[n] = -(y0[j] + sms * H[j]);
        return;
    }
    if (CM == CM_RHS) {
#pragma unroll
        for (int j = 0; j < 3; ++j) comp(a.out, j, nn)[n] = f[j];
    } else if (CM == CM_RK0 || CM == CM_RKS || CM == CM_RKN) {
        const NmRkArgs<T> &r = a.rk;
        T acc[3], ea[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            acc[j] = r.cself * f[j];
            ea[j] = r.eself * f[j];
        }
        T base[3] = {y0[0], y0[1], y0[2]};
        if (CM == CM_RKS) {
#pragma unroll
            for (int j = 0; j < 3; ++j)
                base[j] = r.bs[0] * y0[j] + r.bs[1] * sp[j] + r.bs[2] * sp[3 + j] + r.bs[3] * mc[j];    // sp: the two stage states, loaded with y0
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
#pragma unroll
            for (int j = 0; j < 3; ++j) comp(r.kstore, j, nn)[n] = f[j];
        }
        if (r.ynext) {
            T y[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) y[j] = base[j] + r.dt * acc[j];
            if (r.renorm) {
                const T n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
                const T inv = n2 > (T)0 ? rsqrt_c<T>(n2) : (T)0;   // a zero vector (vacuum node) stays zero
                y[0] *= inv; y[1] *= inv; y[2] *= inv;
            }
#pragma unroll
            for (int j = 0; j < 3; ++j) comp(r.ynext, j, nn)[n] = y[j];
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
#pragma unroll
            for (int j = 0; j < 3; ++j) comp(a.out, j, nn)[n] = f[j];
        }
        const T av[3] = {y0[0], y0[1], y0[2]};
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
            comp(a.dadt, j, nn)[n] = d;
            comp(a.Q, j, nn)[n] = b[j] * invS;
            bH += b[j] * H[j];
        }
        a.W[n] = bH * invS;
    }
}

// Tile geometry (host and device agree through this struct).  Elements per stage:
//   m tiles    3 x (RY + 2) rows x MP: ghost column, n1 nodes, ghost column
//   cell tiles [4 zeros] ncell x (RY + 1) rows x CP: N1 cells, zeros
// The zeros are written once and never touched by the copies: they are cell -1 (the pad of the row
// before) and cell N1 of every cell row.  The row pitches MP = PITCH >= n1 + 2 and CP = PITCH + 4 are
// compile-time (two classes, 264 and 320), so every shared-memory access of the plane arithmetic is
// a base register plus an immediate.
struct ColGeom {
    int MP, CP;
    int moff_cells;         // offset of cell (row 0, column 0) of component 0 in a stage
    int ncell;              // cell tiles per stage: 0 (no demag), 3 (uniform Ms) or 4 (+ Ms)
    int stage;              // elements per stage
    int cvec;               // 1: cell rows are copied in 16-byte pieces
    int cchunks;            // copies per component of the cell tile
};

template <typename T, int RY, int PITCH>
__host__ __device__ inline ColGeom col_geom(const NmGeom &g, bool has_hc, bool uni_ms)
{
    ColGeom c;
    c.MP = PITCH;
    c.CP = PITCH + 4;
    c.moff_cells = ((3 * (RY + 2) * c.MP + 3) / 4) * 4 + 4;
    c.ncell = has_hc ? (uni_ms ? 3 : 4) : 0;
    c.stage = c.moff_cells + c.ncell * (RY + 1) * c.CP;
    c.cvec = ((g.N1 * sizeof(T)) % 16 == 0) ? 1 : 0;
    c.cchunks = c.cvec ? (RY + 1) * (g.N1 / (16 / (int)sizeof(T))) : (RY + 1) * g.N1;
    return c;
}

// TMA-fed form (N1T > 0: the mesh has exactly N1T cells per row, known at compile time).  The RY + 2 node
// rows a CTA needs of one component and plane are (RY + 2)(N1T + 1) contiguous elements of the nodal array:
// the producer thread fetches them with one bulk copy (cp.async.bulk) and each cell row with another; a stage
// completes on an mbarrier.  A bulk copy starts and ends on 16-byte boundaries and node rows do not (n1 is
// odd), so the copy starts at the element index rounded down to a multiple of AL = 4 (fp32) or 2 (fp64) and
// the rows sit `shift` < AL elements into the tile, a number that changes with the plane and the component.
// (A 1-D tensor map was tried first: its boxes must start on 16-byte boundaries too, and fifteen 1 KB boxes
// per plane were slower than three copies.)  Rows keep the array's own pitch n1 = N1T + 1 and there are no ghost columns: the end columns read themselves as
// their missing neighbour (the same mirrored value), and the first / last CTA of the row axis copy the
// mirrored ghost row inside the tile.
template <typename T, int RY, int N1T> struct ColTma {
    static constexpr int n1 = N1T + 1;
    static constexpr int BOX = 256;                                  // elements per box
    static constexpr int AL = 16 / (int)sizeof(T);                   // elements per 16 bytes: copies start and end on these
    static constexpr int NB = ((RY + 2) * n1 + AL - 1 + BOX - 1) / BOX;
    static constexpr int MS = NB * BOX;                              // elements per component tile (rows + shift, rounded)
    static constexpr int CP = N1T + 4;                               // cell row pitch: N1T cells, zeros
    static constexpr int OFF_C = 3 * MS + 4;                         // cell (row 0, column 0) of component 0; 4 zeros before
    __host__ __device__ static constexpr int stage(int ncell) { return ((OFF_C + ncell * (RY + 1) * CP + 31) / 32) * 32; }
};

constexpr int CQ = 3;       // cell copies per thread and component (host checks cchunks <= CQ * threads)

template <typename T, int RY, int CS, int CM, bool UNI_MS, int MAXT, int PITCH, int N1T>
__global__ void __launch_bounds__(MAXT, sizeof(T) == 8 ? 1 : 2)
k_node_col(const NmLocalArgs<T> a, int zchunk)
{
    static_assert(RY == 2, "the plane arithmetic pairs the two node rows of a thread");
    typedef typename PairOf<T>::V V;
    typedef ColTma<T, RY, N1T> TM;
    constexpr bool TMA = N1T > 0;
    extern __shared__ __align__(1024) unsigned char col_smem[];
    T *sm = reinterpret_cast<T *>(col_smem);
    const NmGeom &g = a.g;
    const int n1 = TMA ? TM::n1 : g.n1, n2 = g.n2, N1 = TMA ? N1T : g.N1;
    const bool has_hc = a.Hc != nullptr;
    ColGeom cg = col_geom<T, RY, PITCH>(g, has_hc, UNI_MS);
    if (TMA) {          // the same names, the TMA tile geometry
        cg.CP = TM::CP;
        cg.moff_cells = TM::OFF_C;
        cg.stage = TM::stage(cg.ncell);
    }
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int r0 = blockIdx.x * RY;                       // first node row of the CTA
    const int z0 = blockIdx.y * zchunk, z1 = min(z0 + zchunk, g.n3);
    const unsigned pl = (unsigned)n1 * n2, cpl = (unsigned)N1 * g.N2;
    const size_t nn = (size_t)g.nodes, nc = (size_t)g.cells;
    const bool live = tid < n1;
    constexpr bool RK = CM == CM_RK0 || CM == CM_RKS || CM == CM_RKN;

    for (int q = tid; q < CS * cg.stage; q += nthr) sm[q] = (T)0;
    // TMA: per stage a transaction barrier (the copies have landed) and a barrier the consumer warps arrive on
    // (they have left the stage); warp NW, past the last node column, is the producer
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + CS * cg.stage);
    uint64_t *empty = full + CS;
    const int NW = (n1 + 31) / 32;
    const bool producer = TMA && tid >= NW * 32;
    if (TMA) {
        if (tid == 0) {
            for (int q = 0; q < CS; ++q) {
                mbar_init(full + q, 1);
                mbar_init(empty + q, NW);
            }
            mbar_fence_init();
        }
        fence_async_smem();                                 // the zeros are written before any bulk copy lands
    }
    __syncthreads();

    // ---- what this thread copies every plane (fixed offsets; only the plane base moves) ----------
    // m: column t of every tile row <- node column clamp(t - 1) of node row clamp(r0 - 1 + r)
    const bool mcopy = tid < n1 + 2;
    const unsigned mx = (unsigned)min(max(tid - 1, 0), n1 - 1);
    unsigned mrow[RY + 2];
#pragma unroll
    for (int r = 0; r < RY + 2; ++r) mrow[r] = (unsigned)min(max(r0 - 1 + r, 0), n2 - 1) * n1 + mx;
    // cells: piece e = tid + q nthr of the (RY + 1) x N1 rows, zero-filled where the row does not exist
    unsigned csrc[CQ], cdst[CQ];
    bool cok[CQ], cdo[CQ];
    {
        const int V = cg.cvec ? 16 / (int)sizeof(T) : 1;
        const int per_row = N1 / V;
#pragma unroll
        for (int q = 0; q < CQ; ++q) {
            const int e = tid + q * nthr;
            const int row = e / per_row, ch = e - row * per_row;
            const int c2 = r0 - 1 + row;
            cdo[q] = has_hc && e < cg.cchunks;
            cok[q] = cdo[q] && c2 >= 0 && c2 < g.N2;
            csrc[q] = cok[q] ? (unsigned)c2 * N1 + ch * V : 0u;
            cdst[q] = (unsigned)(cg.moff_cells + row * cg.CP + ch * V);
        }
    }
    const unsigned sm_base = smem_addr(sm);
    // TMA: rows of the cell tile that exist for this CTA (uniform), the same on every plane
    int crow_lo = 0, crow_hi = -1;
    if (TMA && has_hc) {
        crow_lo = r0 - 1 < 0 ? 1 : 0;
        crow_hi = min(RY, g.N2 - r0);                      // tile row `row` is cell row r0 - 1 + row < N2
    }
    auto issue = [&](int k, int slot) {
        if (TMA) {      // the producer thread: three copies of node rows, one per cell row
            T *sb = sm + slot * cg.stage;
            const int kc = min(max(k, 0), g.n3 - 1);
            const bool cv = has_hc && k - 1 >= 0 && k - 1 < g.N3;
            const int E = 3 * (int)nn;
            int e0[3], len[3], off[3], total = cv ? (crow_hi - crow_lo + 1) * (UNI_MS ? 3 : 4) * N1T : 0;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                // rows r0 - 1 .. r0 + RY of component j, plane kc: (RY + 2) n1 contiguous elements from the 16-byte
                // boundary below their start, clipped to the array (what is clipped belongs to rows that do not
                // exist, except the last elements of the array when its length is not a multiple of 4)
                e0[j] = (j * (int)nn + kc * (int)pl + (r0 - 1) * TM::n1) & ~(TM::AL - 1);
                len[j] = ((RY + 2) * TM::n1 + 2 * (TM::AL - 1)) & ~(TM::AL - 1);
                off[j] = 0;
                if (e0[j] < 0) { off[j] = -e0[j]; len[j] += e0[j]; e0[j] = 0; }
                if (e0[j] + len[j] > E) {
                    len[j] = (E - e0[j]) & ~(TM::AL - 1);
                    for (int q = e0[j] + len[j]; q < E; ++q) sb[j * TM::MS + off[j] + q - e0[j]] = a.fld[q];
                }
                total += len[j];
            }
            mbar_expect_tx(full + slot, (uint32_t)(total * sizeof(T)));      // releases the stores above with it
#pragma unroll
            for (int j = 0; j < 3; ++j)
                bulk_load(sb + j * TM::MS + off[j], a.fld + e0[j], (uint32_t)(len[j] * sizeof(T)), full + slot);
            if (cv) {
                const size_t kc2 = (size_t)(k - 1) * cpl;
                for (int j = 0; j < (UNI_MS ? 3 : 4); ++j) {
                    const T *src = (j < 3 ? comp(a.Hc, j, nc) : a.Ms) + kc2;
                    for (int row = crow_lo; row <= crow_hi; ++row)
                        bulk_load(sb + TM::OFF_C + (j * (RY + 1) + row) * TM::CP, src + (size_t)(r0 - 1 + row) * N1T,
                                  (uint32_t)(N1T * sizeof(T)), full + slot);
                }
            }
            return;
        }
        const unsigned sbase = sm_base + (unsigned)(slot * cg.stage) * (unsigned)sizeof(T);
        if (mcopy) {
            const unsigned kc = (unsigned)min(max(k, 0), g.n3 - 1) * pl;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T *src = comp(a.fld, j, nn) + kc;
#pragma unroll
                for (int r = 0; r < RY + 2; ++r) {
                    const unsigned d = sbase + (unsigned)((j * (RY + 2) + r) * cg.MP + tid) * (unsigned)sizeof(T);
                    if (sizeof(T) == 4)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(src + mrow[r]) : "memory");
                    else
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src + mrow[r]) : "memory");
                }
            }
        }
        if (has_hc) {
            const bool cv = k - 1 >= 0 && k - 1 < g.N3;
            const unsigned kc = cv ? (unsigned)(k - 1) * cpl : 0u;
#pragma unroll
            for (int q = 0; q < CQ; ++q) {
                if (!cdo[q]) continue;
                const int sz = (cv && cok[q]) ? (cg.cvec ? 16 : (int)sizeof(T)) : 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (j == 3 && UNI_MS) continue;
                    const T *src = (j < 3 ? comp(a.Hc, j, nc) : a.Ms) + kc + csrc[q];
                    const unsigned d = sbase + (cdst[q] + (unsigned)(j * (RY + 1) * cg.CP)) * (unsigned)sizeof(T);
                    if (cg.cvec)
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
                    else if (sizeof(T) == 4)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
                    else
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
                }
            }
        }
    };

    // ---- per-thread constants -------------------------------------------------------------------------
    // lumped 1-D mass factors of this node column and of the RY rows (1 inside, 1/2 at the two ends;
    // an axis with a single node never occurs: N_d >= 1)
    const T dxf = (tid > 0 && tid < N1) ? (T)1 : (T)0.5;
    const T sixth = (T)(1.0 / 6.0);
    const T c3 = (a.idx2[0] + a.idx2[1]) * sixth;
    const T cUy = a.idx2[1] * dxf, cWy = dxf * sixth;
    T dyf[RY], inv_xy[RY];
    bool rowlive[RY];
#pragma unroll
    for (int ry = 0; ry < RY; ++ry) {
        const int i2 = r0 + ry;
        dyf[ry] = (i2 > 0 && i2 < g.N2) ? (T)1 : (T)0.5;
        rowlive[ry] = live && i2 < n2;
        inv_xy[ry] = UNI_MS ? (T)1 / (a.ms_uni * (T)4 * dxf * dyf[ry]) : (T)0;   // 1 / (S Ms) up to the z factor
    }
    const T cT = UNI_MS ? a.ms_uni : (T)1;

    // pair constants of the plane arithmetic (lo = row r0, hi = row r0 + 1)
    const V DYF = pr<T>(dyf[0], dyf[1]);
    const V kUx = pmul(pr1<T>(a.idx2[0]), DYF);            // dx^-2 dy
    const V kW0 = pmul(pr1<T>(dxf), DYF);                  // dx dy
    const V kW1n = pmul(pr1<T>(-sixth), DYF);              // -dy/6

    // partial sums of the z operators: P waits for the next plane, M starts the output after it
    V GP[3], GM[3], aP, aM;
    aP = aM = pr1<T>((T)0);
#pragma unroll
    for (int j = 0; j < 3; ++j) GP[j] = GM[j] = pr1<T>((T)0);
    double err2 = 0.0;

    const int kstart = max(z0 - 1, 0), kend = z1;         // plane kend = n3 is fetched clamped and weighted 0
    if (!TMA) {
#pragma unroll
        for (int s = 0; s < CS - 2; ++s) {
            if (kstart + s <= kend) issue(kstart + s, s);
            cp_commit();
        }
    } else if (tid == NW * 32) {
        // producer: plane k goes into stage (k - kstart) % CS as soon as every consumer warp has left the plane
        // that used it last; the consumers hold two stages (planes k - 1 and k), so the copies run CS - 2 ahead
        int it = 0;
        for (int k = kstart; k <= kend; ++k, ++it) {
            const int sl = it % CS;
            if (it >= CS) mbar_wait_idle(empty + sl, (uint32_t)((it / CS - 1) & 1));
            issue(k, sl);
        }
    }
    // TMA: x neighbours of the end columns are the columns themselves (mirrored ghosts); tile rows whose node
    // row does not exist are copied from the mirrored one when the stage has landed (first / last CTA only)
    const int xlo = tid > 0 ? -1 : 0, xhi = tid < n1 - 1 ? 1 : 0;
    const bool edge = TMA && (r0 == 0 || r0 + RY > n2 - 1);
    int slot = 0;
    int shc[3] = {0, 0, 0}, shp[3] = {0, 0, 0};            // TMA: shift of the rows in the tiles of plane k and of plane k - 1
    unsigned fphase = 0;                                   // bit q: parity of the next completion of stage q
    unsigned nbase = (unsigned)(kstart - 1) * pl + (unsigned)r0 * n1 + tid;    // node (z = k - 1, row r0, column tid); unused while z < 0
    for (int k = producer ? kend + 1 : kstart; k <= kend; ++k, nbase += pl) {
        if (TMA) {
            const int kc = min(max(k, 0), g.n3 - 1);
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                shp[j] = shc[j];
                shc[j] = (j * (int)nn + kc * (int)pl + (r0 - 1) * TM::n1) & (TM::AL - 1);
            }
            mbar_wait(full + slot, (fphase >> slot) & 1u);
            fphase ^= 1u << slot;
        } else {
            cp_wait<CS - 3>();
            __syncthreads();
            const int kn = k + CS - 2;
            int sn = slot + CS - 2;
            if (sn >= CS) sn -= CS;
            if (kn <= kend) issue(kn, sn);
            cp_commit();
        }
        if (edge) {
            T *sb = sm + slot * cg.stage;
            if (live) {
#pragma unroll
                for (int r = 0; r < RY + 2; ++r) {
                    const int i2 = r0 - 1 + r;
                    const int ic = min(max(i2, 0), n2 - 1);
                    if (ic != i2) {
#pragma unroll
                        for (int j = 0; j < 3; ++j)
                            sb[j * TM::MS + shc[j] + r * TM::n1 + tid] = sb[j * TM::MS + shc[j] + (ic - (r0 - 1)) * TM::n1 + tid];
                    }
                }
            }
            fence_async_smem();
            asm volatile("bar.sync 1, %0;" ::"r"(NW * 32) : "memory");     // the consumer warps only
        }
        const int z = k - 1;
        const bool zout = z >= z0 && z < z1;
        // what the epilogue reads at its nodes (start-of-step state, a, or d): loaded now, used after
        // the plane arithmetic
        T y0[RY][3], ys[RY][CM == CM_RKS ? 6 : 1];
        if ((RK || CM == CM_ADJ1 || CM == CM_ADJ2) && zout) {
            const T *pre = RK ? a.rk.y0 : (CM == CM_ADJ1 ? a.adj : a.dadt);
#pragma unroll
            for (int ry = 0; ry < RY; ++ry)
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    y0[ry][j] = rowlive[ry] ? comp(pre, j, nn)[nbase + ry * n1] : (T)0;
                    if (CM == CM_RKS) {     // last RK4 stage: the two stage states it combines, too (their latency was the epilogue's)
                        ys[ry][j] = rowlive[ry] ? comp(a.rk.sprev[0], j, nn)[nbase + ry * n1] : (T)0;
                        ys[ry][3 + j] = rowlive[ry] ? comp(a.rk.sprev[1], j, nn)[nbase + ry * n1] : (T)0;
                    }
                }
        }
        // plane-uniform z coefficients: plane k is the centre of output k, the upper neighbour of
        // output k - 1 and the lower neighbour of output k + 1
        const T gLk = k > 0 ? (T)1 : (T)0, gRk = k < g.N3 ? (T)1 : (T)0;      // of output k
        const T gRm = (k - 1 < g.N3) ? (T)1 : (T)0;                           // gR of output k - 1
        const T gLp = (T)1;                                                   // gL of output k + 1
        const T dzk = (T)0.5 * (gLk + gRk);
        const T eR_out = a.cex * gRm;                     // -cex * (-gR R_k)
        const T eU_P = -a.cex * dzk, eR_P = -a.cex * (gLk + gRk);
        const T eR_M = a.cex * gLp;
        const T wR_out = gRm * sixth, w_P = dzk - (gLk + gRk) * sixth, w_M = gLp * sixth;
        const T *st = sm + slot * cg.stage;
        // TMA: a cell plane that does not exist is not fetched (the stage keeps older, finite values): weight 0
        const T cTk = (TMA && !(k - 1 >= 0 && k - 1 < g.N3)) ? (T)0 : cT;
        if (live) {
            V Tn[3];
            if (has_hc) {
                const T *cb = st + cg.moff_cells + tid;
                T ml[RY + 1], mr[RY + 1];
                if (!UNI_MS) {
#pragma unroll
                    for (int cr = 0; cr < RY + 1; ++cr) {
                        const T *mrow_ = cb + (3 * (RY + 1) + cr) * cg.CP;
                        ml[cr] = mrow_[-1];
                        mr[cr] = mrow_[0];
                    }
                }
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    T X[RY + 1];
#pragma unroll
                    for (int cr = 0; cr < RY + 1; ++cr) {
                        const T *crow = cb + (j * (RY + 1) + cr) * cg.CP;
                        X[cr] = UNI_MS ? crow[-1] + crow[0] : ml[cr] * crow[-1] + mr[cr] * crow[0];
                    }
                    Tn[j] = pmul(pr1<T>(cTk), padd(pr<T>(X[0], X[1]), pr<T>(X[1], X[2])));
                }
            } else {
                Tn[0] = Tn[1] = Tn[2] = pr1<T>((T)0);
            }
            V wk = pr1<T>((T)0);
            V Gout[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                T c[RY + 2], sx[RY + 2];
                if (TMA) {
                    const T *t = st + j * TM::MS + shc[j] + tid;  // rows at the array's pitch, no ghost columns
#pragma unroll
                    for (int r = 0; r < RY + 2; ++r) {
                        c[r] = t[r * TM::n1];
                        sx[r] = (t + xlo)[r * TM::n1] + (t + xhi)[r * TM::n1];
                    }
                } else {
                    const T *t = st + j * (RY + 2) * cg.MP + tid; // columns tid, tid + 1, tid + 2 = i1 - 1, i1, i1 + 1
#pragma unroll
                    for (int r = 0; r < RY + 2; ++r) {
                        const T *row = t + r * cg.MP;
                        c[r] = row[1];
                        sx[r] = row[0] + row[2];
                    }
                }
                const V CC = pr<T>(c[1], c[2]), SXc = pr<T>(sx[1], sx[2]);
                const V ax = pfma(CC, pr1<T>((T)2), pneg(SXc));
                const V ay = pfma(CC, pr1<T>((T)2), pneg(padd(pr<T>(c[0], c[1]), pr<T>(c[2], c[3]))));
                const V axy = pfma(padd(ax, ay), pr1<T>((T)2),
                                   pfma(CC, pr1<T>((T)-4), padd(pr<T>(sx[0], sx[1]), pr<T>(sx[2], sx[3]))));
                const V U = pfma(kUx, ax, pfma(ay, pr1<T>(cUy), pmul(axy, pr1<T>(-c3))));
                const V W = pfma(kW0, CC, pfma(kW1n, ax, pfma(ay, pr1<T>(-cWy), pmul(axy, pr1<T>((T)(1.0 / 36.0))))));
                const V R = pfma(W, pr1<T>(a.idx2[2]), pmul(U, pr1<T>(-sixth)));
                wk = pfma(W, pr1<T>(a.kax[j]), wk);
                Gout[j] = padd(pfma(R, pr1<T>(eR_out), GP[j]), Tn[j]);
                GP[j] = padd(pfma(R, pr1<T>(eR_P), pfma(U, pr1<T>(eU_P), GM[j])), Tn[j]);
                GM[j] = pmul(R, pr1<T>(eR_M));
            }
            const V aout = pfma(wk, pr1<T>(wR_out), aP);
            aP = pfma(wk, pr1<T>(w_P), aM);
            aM = pmul(wk, pr1<T>(w_M));
            if (zout) {
                const T gLz = z > 0 ? (T)1 : (T)0;
                const T izf = (z > 0 && z < g.N3) ? (T)0.5 : (T)1;             // 1 / (gL + gR) of output z
                int sp = slot - 1;
                if (sp < 0) sp += CS;
                const T *sprev = sm + sp * cg.stage + tid + (TMA ? 0 : 1);    // centre column of plane z
                const unsigned nrow[RY] = {nbase, nbase + (unsigned)n1};
                V mcp[3];
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    mcp[j] = TMA ? pr<T>(sprev[j * TM::MS + shp[j] + TM::n1], sprev[j * TM::MS + shp[j] + 2 * TM::n1])
                                 : pr<T>(sprev[(j * (RY + 2) + 1) * cg.MP], sprev[(j * (RY + 2) + 2) * cg.MP]);
                V smsp, invp;
                if (UNI_MS) {
                    invp = pmul(pr<T>(inv_xy[0], inv_xy[1]), pr1<T>(izf));
                    smsp = (CM == CM_ADJ1 || CM == CM_ADJ2) ? pmul(DYF, pr1<T>(a.ms_uni * (T)4 * dxf * (gLz + gRm))) : pr1<T>((T)1);
                } else {
                    smsp = pr<T>(rowlive[0] ? a.sMs[nrow[0]] : (T)0, rowlive[1] ? a.sMs[nrow[1]] : (T)0);
                    invp = pr<T>(smsp.x > 0 ? rcp_c<T>(smsp.x) : (T)0, smsp.y > 0 ? rcp_c<T>(smsp.y) : (T)0);
                }
                // H = (anisotropy + exchange + demag sums) / (S Ms) + uniform Zeeman; 0 where S Ms = 0
                const V ak = pmul(aout, pr1<T>(a.cku));
                V Hp[3];
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    Hp[j] = pmul(pfma(ak, pr1<T>(a.kax[j]), Gout[j]), invp);
                    if (a.terms & NM_TERM_ZEEMAN) {
                        const T hz = a.hu[j];
                        Hp[j] = padd(Hp[j], UNI_MS ? pr1<T>(hz) : pr<T>(smsp.x > 0 ? hz : (T)0, smsp.y > 0 ? hz : (T)0));
                    }
                    if (a.hadd)     // smoothed nodal Zeeman field and / or the further local terms (0 where S Ms = 0)
                        Hp[j] = padd(Hp[j], pr<T>(rowlive[0] ? comp(a.hadd, j, nn)[nrow[0]] : (T)0,
                                                  rowlive[1] ? comp(a.hadd, j, nn)[nrow[1]] : (T)0));
                }
                // a9 (Eq. 1) on both rows: f = -gamma' m x H - alpha gamma' m x (m x H)
                V fp[3];
                if (CM != CM_H && CM != CM_ADJ2) {
                    V mxH[3], mm[3];
                    mxH[0] = pfma(mcp[1], Hp[2], pneg(pmul(mcp[2], Hp[1])));
                    mxH[1] = pfma(mcp[2], Hp[0], pneg(pmul(mcp[0], Hp[2])));
                    mxH[2] = pfma(mcp[0], Hp[1], pneg(pmul(mcp[1], Hp[0])));
                    mm[0] = pfma(mcp[1], mxH[2], pneg(pmul(mcp[2], mxH[1])));
                    mm[1] = pfma(mcp[2], mxH[0], pneg(pmul(mcp[0], mxH[2])));
                    mm[2] = pfma(mcp[0], mxH[1], pneg(pmul(mcp[1], mxH[0])));
#pragma unroll
                    for (int j = 0; j < 3; ++j) fp[j] = pfma(mxH[j], pr1<T>(-a.gp), pmul(mm[j], pr1<T>(-a.agp)));
                } else {
                    fp[0] = fp[1] = fp[2] = pr1<T>((T)0);
                }
#pragma unroll
                for (int ry = 0; ry < RY; ++ry) {
                    if (!rowlive[ry]) continue;
                    const T mc[3] = {ry ? mcp[0].y : mcp[0].x, ry ? mcp[1].y : mcp[1].x, ry ? mcp[2].y : mcp[2].x};
                    const T H[3] = {ry ? Hp[0].y : Hp[0].x, ry ? Hp[1].y : Hp[1].x, ry ? Hp[2].y : Hp[2].x};
                    const T f[3] = {ry ? fp[0].y : fp[0].x, ry ? fp[1].y : fp[1].x, ry ? fp[2].y : fp[2].x};
                    epilogue_c<T, CM>(a, nrow[ry], nn, mc, H, f, ry ? smsp.y : smsp.x, y0[ry], ys[ry], err2);
                }
            }
        }
        if (TMA && k > kstart) {          // plane k - 1 is no longer needed by this warp
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(empty + (slot == 0 ? CS - 1 : slot - 1));
        }
        if (++slot == CS) slot = 0;
    }
    if (!TMA) cp_wait<0>();
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
inline int col_threads(const NmGeom &g) { return ((g.n1 + 2 + 31) / 32) * 32; }

// pitch class of a mesh: the smaller compile-time row pitch that holds n1 + 2 columns
constexpr int kPitchS = 264, kPitchL = 320;
inline int col_pitch(const NmGeom &g) { return g.n1 + 2 <= kPitchS ? kPitchS : kPitchL; }
template <typename T> inline ColGeom col_geom_rt(const NmGeom &g, bool has_hc, bool uni_ms)
{
    return col_pitch(g) == kPitchS ? col_geom<T, kRY, kPitchS>(g, has_hc, uni_ms) : col_geom<T, kRY, kPitchL>(g, has_hc, uni_ms);
}

template <typename T, int CM, bool UNI_MS, int PITCH>
nm_status launch_col_p(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    constexpr int CS = ColStages<T>::CS;
    const NmGeom &g = a.g;
    const ColGeom cg = col_geom<T, kRY, PITCH>(g, a.Hc != nullptr, UNI_MS);
    const size_t bytes = (size_t)CS * cg.stage * sizeof(T);
    const int zchunk = col_zchunk(g);
    const dim3 grid((g.n2 + kRY - 1) / kRY, (g.n3 + zchunk - 1) / zchunk);
    auto kern = k_node_col<T, kRY, CS, CM, UNI_MS, kMaxT, PITCH, 0>;
    NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    mesh->last_partials = (int)(grid.x * grid.y);
    {
        NmLaunchScope sc(mesh, nm_node_class(a.mode), st);
        kern<<<grid, col_threads(g), bytes, st>>>(a, zchunk);
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

// ---- TMA-fed form: N1 = 128 or 256 cells per row ----------------------------------------------------------
// which compile-time row length serves this launch (0: the cp.async form)
template <typename T> int col_tma_n1(const nm_mesh *mesh, const NmLocalArgs<T> &a)
{
    if (mesh->dbg_node_path == 3) return 0;                // NM_NODE_PATH=ring at nm_mesh_create (tests, measurements)
    const NmGeom &g = a.g;
    if (g.N1 != 128 && g.N1 != 256) return 0;
    if (3 * g.nodes >= (1ll << 31) || (((uintptr_t)a.fld) & 15)) return 0;
    if (a.Hc && ((((uintptr_t)a.Hc) | ((uintptr_t)a.Ms)) & 15)) return 0;
    return g.N1;
}

template <typename T, int CM, bool UNI_MS, int N1T>
nm_status launch_col_tma(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    constexpr int CS = ColStages<T>::CS;
    typedef ColTma<T, kRY, N1T> TM;
    const NmGeom &g = a.g;
    const int ncell = a.Hc ? (UNI_MS ? 3 : 4) : 0;
    const size_t bytes = (size_t)CS * TM::stage(ncell) * sizeof(T) + 2 * CS * sizeof(uint64_t);
    const int zchunk = col_zchunk(g);
    const dim3 grid((g.n2 + kRY - 1) / kRY, (g.n3 + zchunk - 1) / zchunk);
    auto kern = k_node_col<T, kRY, CS, CM, UNI_MS, kMaxT, kPitchS, N1T>;
    NM_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    mesh->last_partials = (int)(grid.x * grid.y);
    {
        NmLaunchScope sc(mesh, nm_node_class(a.mode), st);
        kern<<<grid, ((TM::n1 + 31) / 32 + 1) * 32, bytes, st>>>(a, zchunk);      // + the producer warp
    }
    NM_CUDA_TRY(cudaGetLastError());
    return NM_OK;
}

template <typename T, int CM, bool UNI_MS>
nm_status launch_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    const int nt = col_tma_n1<T>(mesh, a);
    if (nt == 256) return launch_col_tma<T, CM, UNI_MS, 256>(mesh, a, st);
    if (nt == 128) return launch_col_tma<T, CM, UNI_MS, 128>(mesh, a, st);
    return col_pitch(a.g) == kPitchS ? launch_col_p<T, CM, UNI_MS, kPitchS>(mesh, a, st)
                                     : launch_col_p<T, CM, UNI_MS, kPitchL>(mesh, a, st);
}

template <typename T, bool UNI_MS> nm_status dispatch_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st)
{
    switch (a.mode) {
    case NM_MODE_H: return launch_col<T, CM_H, UNI_MS>(mesh, a, st);
    case NM_MODE_RHS: return launch_col<T, CM_RHS, UNI_MS>(mesh, a, st);
    case NM_MODE_ADJ1: return launch_col<T, CM_ADJ1, UNI_MS>(mesh, a, st);
    case NM_MODE_ADJ2: return launch_col<T, CM_ADJ2, UNI_MS>(mesh, a, st);
    default:
        if (!a.rk.want_err && a.rk.nprev == 0 && a.rk.nstate == 0) return launch_col<T, CM_RK0, UNI_MS>(mesh, a, st);
        if (!a.rk.want_err && a.rk.nprev == 0 && a.rk.nstate == 2) return launch_col<T, CM_RKS, UNI_MS>(mesh, a, st);
        return launch_col<T, CM_RKN, UNI_MS>(mesh, a, st);
    }
}

} // namespace

// Eligibility: the separable operators (uniform A, Ku; no nodal Zeeman arrays -- decided by the
// caller), a thread per node column plus the two ghost columns, 32-bit node indices, and a ring of
// stages that fits the shared memory of an SM (two CTAs per SM in fp32).
template <typename T> bool nm_node_col_ok(const nm_mesh *mesh, const NmLocalArgs<T> &a)
{
    (void)mesh;
    const NmGeom &g = a.g;
    if (g.n1 < 96 || g.n1 + 2 > kMaxT || g.nodes >= (1ll << 31)) return false;
    const ColGeom cg = col_geom_rt<T>(g, a.Hc != nullptr, a.ms_uni > 0);
    if (cg.cchunks > CQ * col_threads(g)) return false;
    if (cg.cvec && a.Hc && ((((uintptr_t)a.Hc) | ((uintptr_t)a.Ms)) & 15)) return false;   // 16-byte cell copies
    const size_t bytes = (size_t)ColStages<T>::CS * cg.stage * sizeof(T);
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
