// Argument blocks of the node / cell kernels in nm_local.cu (internal).
#pragma once

#include "nm_internal.h"

enum NmLocalMode {
    NM_MODE_H = 0,      // out = H_eff
    NM_MODE_RHS = 1,    // out = f(m, H)                                  (Eq. 1)
    NM_MODE_RK = 2,     // Runge-Kutta stage epilogue (a10)
    NM_MODE_ADJ1 = 3,   // adjoint pass 1: f, b, d, q = b/(S Ms), w = b.H/(S Ms)
    NM_MODE_ADJ2 = 4    // adjoint pass 2: dadt = -(d + (S Ms) Hlin(q))
};

template <typename T> struct NmRkArgs {
    const T *y0;        // state at the start of the step
    T *kstore;          // where to keep this stage's derivative (or null)
    const T *kprev[6];  // earlier stage derivatives
    T cprev[6];         // their weights in the next stage state / final update
    T eprev[6];         // their weights in the embedded error (last Dormand-Prince stage)
    int nprev;
    T cself, eself;
    // nstate = 2: last stage of RK4 from the stage states (no stored derivatives): with
    // Y0 = y + dt/2 k1, Y1 = y + dt/2 k2 and fld = y + dt k3,
    //   ynext = bs[0] y0 + bs[1] sprev[0] + bs[2] sprev[1] + bs[3] fld + dt cself f
    const T *sprev[2];
    T bs[4];
    int nstate;
    T *ynext;           // y0 + dt (sum cprev kprev + cself f), or null
    T dt;
    int renorm;         // normalise ynext (final RK4 update written to m in place)
    int want_err;       // accumulate the scaled squared error into partials[blockIdx.x]
    T rtol, atol;
    double *partials;
};

template <typename T> struct NmLocalArgs {
    NmGeom g;
    const T *fld;       // nodal field the linear operators act on (m, or q in NM_MODE_ADJ2)
    const T *Ms, *A, *Ku, *sMs;
    const T *Hc;        // cell demag field [3][cells] or null
    unsigned terms;
    T wK[8], wM[8];     // element matrix entries by offset pattern e (bit d: vertices differ along d)
    T kax[3];
    T mu0V8;            // mu0 V / 8
    T mu0;
    // Zeeman: H_ext = hu + h_static + amp * h_pulse
    const T *h_static, *h_pulse;
    T amp;
    T hu[3];
    const T *hadd;      // nodal field added to H as it stands (the smoothed nodal Zeeman field, k_zeeman_smooth), or null
    // LLG
    T gp, agp;          // gamma' = gamma/(1+alpha^2), alpha gamma'
    int mode;
    T *out;             // H (MODE_H), f (MODE_RHS / ADJ1, may be null), dadt (ADJ1: d, ADJ2: final)
    // adjoint
    const T *adj;       // a
    T *Q, *W, *dadt;
    NmRkArgs<T> rk;
    // separable kernel k_node_sep (uniform A and Ku, no nodal Zeeman arrays)
    int sep;            // 0: 27-point kernel; 1: separable kernels (column-marching where it applies); 2: k_node_sep only
    T cex, cku;         // 16 A / mu0 and 16 Ku / mu0 (0 when the term is off)
    T idx2[3];          // 1 / dx_d^2
    T ms_uni;           // > 0: Ms has this value in every cell; 0: read the Ms / sMs arrays
};

template <typename T> struct NmAdjCellArgs {
    NmGeom g;
    const T *m, *Q, *W, *Hc1, *Hc2;
    const T *h_static, *h_pulse;
    T amp;
    T hu[3];
    T wM8V[8];          // (8/V) * mass matrix entry by offset pattern
    T red;              // 2^(D-3): 1 on the 3-D basis (nm_red_scale)
    unsigned terms;
    T *dudt;
};

// Further local terms (NM_TERM_DMI, NM_TERM_CUBIC) evaluated per node into a nodal field that
// the node kernels add to H (NmLocalArgs.hadd)
template <typename T> struct NmExtraArgs {
    NmGeom g;
    const T *fld, *Ms, *D, *Kc;     // nodal m; cell-wise Ms, D, Kc (D / Kc null when the term is off)
    const T *about;                 // null: cubic term = its field at fld; else its linearisation about this nodal m, applied to fld
    T *out;                         // nodal vector: -(dE_dmi + dE_cubic) / L, 0 where (S Ms)_n = 0
    T mu0V8, V;
    T idx[3];                       // 1 / dx_d
    int dmi_kind, dmi_normal;
    T cax[9];                       // cubic frame, rows c_1, c_2, c_3
    T rkky_JA;                      // J dx dy (0: term off)
    int rkky_za, rkky_zb;
};
template <typename T> nm_status nm_launch_extra(nm_mesh *mesh, const NmExtraArgs<T> &a, cudaStream_t st);

// host launchers defined in nm_local.cu
template <typename T> nm_status nm_launch_node(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st);
// nm_node_col.cu: column-marching form of the separable kernel (cp.async stage ring)
template <typename T> bool nm_node_col_ok(const nm_mesh *mesh, const NmLocalArgs<T> &a);
template <typename T> nm_status nm_launch_node_col(nm_mesh *mesh, const NmLocalArgs<T> &a, cudaStream_t st);
int nm_node_col_blocks(const NmGeom &g);
int nm_node_blocks(const NmGeom &g);   // capacity needed for the error-norm partials
nm_status nm_launch_err_final(nm_mesh *mesh, int n_partials, double count, cudaStream_t st);
template <typename T>
nm_status nm_launch_commit(nm_mesh *mesh, T *m, const T *y5, const double *err, int renorm, cudaStream_t st);
template <typename T> nm_status nm_launch_adj_cell(nm_mesh *mesh, const NmAdjCellArgs<T> &a, cudaStream_t st);
// u_h[j] += coef * ( - sum over nodes with (S Ms)_n > 0 of b_n[j] ),  b = g' m x a - alpha g' m x (m x a):
// -(df/dh)^T a for a uniform external field h, accumulated in
// fp64 in a fixed summation order.
template <typename T>
nm_status nm_launch_hext_grad(nm_mesh *mesh, const T *m, const T *a, double gp, double agp, double coef,
                              double *u_h, cudaStream_t st);

// u_hn (+)= coef (-(df/dh)^T a) for a nodal external field h through the weak form:
// the transposed Zeeman smoothing applied to q = b / (S Ms); q = null: made from (m, a) into mesh->Q.
template <typename T>
nm_status nm_launch_hnodal_grad(nm_mesh *mesh, const NmLocalArgs<T> &base, const T *q, const T *m, const T *av,
                                double coef, int accumulate, T *u_hn, cudaStream_t st);

// Cell-wise VJPs with respect to A_c and Ku_c, b = g' m x a - alpha g' m x (m x a),
// bL = b / L (0 where (S Ms)_n = 0), the element matrices K, M of Eq. (12) by vertex difference pattern:
//   gA_c  = +2 sum_{i,i'} K[i,i'] bL_{c+i} . m_{c+i'}           = -(df/dA_c)^T a
//   gKu_c = -2 sum_{i,i'} M[i,i'] (bL_{c+i}.k) (m_{c+i'}.k)     = -(df/dKu_c)^T a
// accumulate == 0: u_X = gX; else u_X += coef gX.  u_A / u_Ku may be null; a term that is off gives 0.
template <typename T> struct NmMatGradArgs {
    NmGeom g;
    const T *m, *a, *sMs;
    T *u_A, *u_Ku;
    T wK[8], wM[8], kax[3];
    T gp, agp, invL;        // invL = 8 / (mu0 V): bL = b invL / (S Ms)
    T coef;
    int accumulate, ex_on, an_on;
};
template <typename T> nm_status nm_launch_mat_grad(nm_mesh *mesh, const NmMatGradArgs<T> &a, cudaStream_t st);

// several independent updates out = base + coef * src in one launch (vec_n > 0: [3][vec_n] arrays,
// result normalised per node); no update may read what another one writes
enum { NM_LIN_OPS = 5 };
template <typename T> struct NmLinOp {
    T *out;
    const T *base, *src;
    T coef;
    long long n, vec_n;
};
template <typename T>
nm_status nm_lincomb_batch(nm_mesh *mesh, const NmLinOp<T> *ops, int nops, cudaStream_t st);

template <typename T>
nm_status nm_lincomb(nm_mesh *mesh, T *out, const T *base, int nsrc, const T *const *src, const T *coef,
                     long long n, long long vec_n, cudaStream_t st);
