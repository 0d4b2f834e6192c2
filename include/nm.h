/* nm.h — C-ABI of the B200-native nodal finite-difference LLG right-hand side.
 *
 * The method is the hot path of NeuralMag (arxiv 2411.11725; citations are lines of
 * /root/reference/PAPER.md): the Landau-Lifshitz-Gilbert right-hand side, Eq. (1),
 * on a nodal finite-difference mesh (magnetisation m on the (N1+1)(N2+1)(N3+1) vertices, material
 * parameters on the N1 N2 N3 cells; Eqs. 8-16) with
 *   - exchange, uniaxial-anisotropy and Zeeman fields from the mass-lumped weak form
 *     (Eqs. 17-22),
 *   - the demagnetisation field as a zero-padded FFT convolution over cells with node<->cell
 *     averaging before and after (Sec. III B),
 *   - explicit Runge-Kutta steps (RK4, Dormand-Prince),
 *   - the adjoint (vector-Jacobian) right-hand side of the adjoint-state system, Eq. (29)
 *     (PAPER.md:219-228).
 * Where the paper is silent the readings C1..C8 of DESIGN.md apply.
 *
 * Conventions
 *   Precision    every array of one mesh has the mesh's dtype (NM_F32: float, NM_F64: double).
 *   Memory       every `const void*` / `void*` array argument is DEVICE memory on `desc.device`
 *                unless the name ends in `_host`.  The caller owns all of it, including the
 *                workspace block handed to nm_mesh_create; the library allocates no device
 *                memory after nm_mesh_create returns and frees none that it did not allocate.
 *   Layout       nodal vector fields are structure-of-arrays [3][N3+1][N2+1][N1+1], x (index 1 of
 *                the paper's multi-index) fastest, contiguous (no row padding).  Nodal scalars [N3+1][N2+1][N1+1].
 *                Cell scalars [N3][N2][N1], cell vectors [3][N3][N2][N1].
 *   Units        SI: H and Ms in A/m, A in J/m, Ku in J/m^3, gamma in m/(A s), t in s
 *                (PAPER.md:37).  mu0 = 4 pi 1e-7 exactly.
 *   Streams      `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All
 *                work is enqueued on it and the call returns without synchronising, except where
 *                stated.  Calls on one mesh must not overlap (they share the workspace).
 *   Errors       every entry point returns nm_status; nothing throws across the ABI;
 *                nm_last_error() returns a thread-local message for the last failure.
 *                NaN/Inf in inputs are not checked.  Nodes all of whose adjacent cells have
 *                Ms = 0 get H = 0 (reading C3(iii)).
 */
#ifndef NM_H
#define NM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nm_mesh nm_mesh; /* opaque, library-owned host object */

typedef enum { NM_F32 = 0, NM_F64 = 1 } nm_dtype;

typedef enum {
    NM_OK = 0,
    NM_EINVAL = -1,       /* bad argument (null pointer, non-positive size, ...) */
    NM_EUNSUPPORTED = -2, /* valid request this build cannot serve (see nm_mesh_create) */
    NM_ECUDA = -3,        /* a CUDA runtime call or kernel launch failed */
    NM_ENOMEM = -4        /* workspace too small / host allocation failed */
} nm_status;

/* field terms, OR-ed into nm_mesh_desc.terms */
enum { NM_TERM_EXCHANGE = 1, NM_TERM_DEMAG = 2, NM_TERM_ANISO = 4, NM_TERM_ZEEMAN = 8,
       /* further local terms through the same weak form ("crystalline anisotropies, and both
          symmetric and antisymmetric exchange interactions", readings F3) */
       NM_TERM_DMI = 16,   /* antisymmetric exchange, density D sum T[a,d,b] m_a d_d m_b (nm_mesh_desc.dmi_kind) */
       NM_TERM_CUBIC = 32, /* cubic anisotropy, density Kc (a1^2 a2^2 + a2^2 a3^2 + a3^2 a1^2), a_q = m . c_q */
       NM_TERM_RKKY = 64   /* interlayer coupling E = -J int m(x,y,z_a) . m(x,y,z_b) dGamma between two node planes
                              (PAPER.md:79), through the 2-D face mass matrix; linear in m: every entry point */
};
typedef enum { NM_DMI_BULK = 0,        /* D m . curl m */
               NM_DMI_INTERFACIAL = 1  /* D [m_n div m - (m . grad) m_n], n = nm_mesh_desc.dmi_normal */
} nm_dmi_kind;

typedef enum { NM_RK4 = 0, NM_DOPRI5 = 1 } nm_scheme;

/* Statement of the problem: regular grid, nodal m, cell-wise materials. */
typedef struct {
    int n_cells[3];       /* N1, N2, N3 >= 1.  With NM_TERM_DEMAG every N_d > 1 must be
                             2^a 3^b 5^c 7^d (FFT radices 2,3,4,5,7,8), else NM_EUNSUPPORTED -- except
                             meshes the zero-extended fast path serves (2 <= N_d <= 256 that
                             fill half of the (y, z) plane of the next sizes 16 * 2^k and
                             meet its row granularities; see nm_debug_demag_path), any N_d. */
    double cell_size[3];  /* metres, > 0 */
    nm_dtype dtype;
    int device;           /* CUDA device ordinal */
    unsigned terms;       /* OR of NM_TERM_* */
    double gamma;         /* reduced gyromagnetic ratio, m/(A s) */
    double alpha;         /* Gilbert damping, scalar */
    double ku_axis[3];    /* anisotropy axis k, unit vector, global (reading C3(i)) */
    const void *Ms, *A, *Ku; /* device, cell-wise [N3][N2][N1], copied at create; NULL => scalar below */
    double Ms_scalar, A_scalar, Ku_scalar;
    int basis;            /* dimensions the nodal basis varies in (Sec. III C):
                             0 or 3  full 3-D nodal basis, (N1+1)(N2+1)(N3+1) nodes;
                             2       film: basis functions constant along z (Eq. 23), needs N3 = 1;
                                     nodal arrays are [3][1][N2+1][N1+1];
                             1       rod: constant along y and z (Eq. 24), needs N2 = N3 = 1; nodal
                                     arrays are [3][1][1][N1+1].
                             The weak form is still integrated over the 3-D cells (element matrices
                             without derivatives along the reduced axes, lumped mass V / 2^D per cell,
                             node <-> cell averaging over the 2^D vertices of a cell).  Every entry
                             point serves the reduced bases, the adjoint ones included. */
    /* NM_TERM_DMI / NM_TERM_CUBIC (3-D basis).  Both are carried by every entry point (the adjoint ones give
       d/dm and d/dMs, not d/dD or d/dKc): the DMI term is linear in m like the exchange term; for the cubic
       term the adjoint right-hand side applies the Hessian of its energy at m.  The element contributions are
       integrated exactly (DMI: bilinear in the Q1 functions; cubic: 3-point Gauss per axis), summed into
       the nodes and divided by the lumped mass, Eqs. (17)-(22). */
    const void *D, *Kc;   /* device, cell-wise [N3][N2][N1], copied at create; NULL => scalar below */
    double D_scalar;      /* J/m^2 */
    double Kc_scalar;     /* J/m^3 */
    int dmi_kind;         /* nm_dmi_kind */
    int dmi_normal;       /* film normal axis (0, 1, 2) of NM_DMI_INTERFACIAL */
    double cubic_axes[9]; /* rows c_1, c_2, c_3: one global orthonormal frame */
    double rkky_J;        /* J/m^2 (NM_TERM_RKKY); > 0 favours parallel layers */
    int rkky_planes[2];   /* node-plane indices z_a != z_b along axis 3, 0 <= z <= N3 */
} nm_mesh_desc;

/* Bytes of device workspace nm_mesh_create needs for this description (spectrum buffers, demag
 * tensor, lumped mass, Runge-Kutta and adjoint scratch).  Host-only call. */
nm_status nm_mesh_query_workspace(const nm_mesh_desc *desc, size_t *bytes_out);

/* Build a mesh object inside the caller's workspace (256-byte aligned device block of at least the
 * queried size).  Computes the demag tensor of uniformly magnetised cuboids (reading C4: Newell
 * closed form in __float128 near the origin, 6-D Gauss quadrature of the dipole kernel beyond
 * 8 cell sizes; both agree with the closed form to < 1e-15), its real, symmetric spectrum with
 * 1/(P1 P2 P3) folded in, S Ms and the FFT tables.  Synchronous; not part of the hot path.
 * Environment switches, read here (and by nm_mesh_query_workspace) once, for tests and measurements; none changes a
 * result beyond rounding: NM_DEMAG_PATH=generic (general-size demag kernels), NM_PIPE=0 (one-CTA-per-tile fast
 * kernels), NM_KT_CHUNK=c (k1 tiles per y/z/y launch group), NM_NODE_PATH=generic|sep|ring (forms of the node
 * kernel), NM_GRAPH=0|1 (whole-step launch replay), NM_FAST192=1 (an axis of 192 cells transformed at its own
 * length, 3 x 64, instead of zero-extended to 256; slower). */
nm_status nm_mesh_create(nm_mesh **out, const nm_mesh_desc *desc, void *workspace, size_t bytes);

/* Replace the cell-wise saturation magnetisation (device array) and recompute S Ms. */
nm_status nm_mesh_set_Ms(nm_mesh *mesh, const void *Ms, void *stream);

/* Frees the host object only (the workspace stays the caller's). */
nm_status nm_mesh_destroy(nm_mesh *mesh);

/* Thread-local message describing the last non-NM_OK status returned on this thread. */
const char *nm_last_error(void);

/* External (Zeeman) field  H_ext(t, n) = h_uniform + h_static[n] + amp(t) * h_pulse[n]
 * (nodal field through the weak form, Eq. 21; reading C3(ii)). */
typedef struct {
    const void *h_static, *h_pulse; /* device nodal 3-vector fields or NULL */
    double h_uniform[3];            /* A/m, added at every node */
    double (*amp)(double t, void *user); /* host callback, called once per field evaluation
                                            (per RK stage) on the calling thread; NULL => 1 */
    void *user;
} nm_zeeman;

/* a1-a8: H_out = H_ex + H_an + H_zeeman + H_demag at the nodes (terms selected at create).
 * `zeeman` may be NULL (no external field). */
nm_status nm_heff(nm_mesh *mesh, double t, const void *m, const nm_zeeman *zeeman, void *H_out,
                  void *stream);

/* a1-a9: dmdt_out = -g' m x H - alpha g' m x (m x H), g' = gamma/(1+alpha^2)  (Eq. 1). */
nm_status nm_llg_rhs(nm_mesh *mesh, double t, const void *m, const nm_zeeman *zeeman,
                     void *dmdt_out, void *stream);

/* a10: one explicit Runge-Kutta step of size dt on m_inout (in place).
 *   NM_RK4     classical tableau, 4 right-hand sides; err_norm_host must be NULL or is set to 0.
 *   NM_DOPRI5  Dormand-Prince 5(4), 7 right-hand sides; the scaled RMS error
 *              err = sqrt(mean(((y5-y4)/(atol + rtol max(|y0|,|y5|)))^2)) over all 3*nodes
 *              components is computed on the device; the step is committed iff err <= 1,
 *              otherwise m_inout is left unchanged.  If err_norm_host != NULL the stream is
 *              synchronised once and *err_norm_host = err (the caller adapts dt).
 *   renormalise != 0: m_n <- m_n/|m_n| once per committed step (reading C6); stages see the
 *              un-normalised intermediate states.
 * Launch replay: on meshes of at most 2^21 cells (launch-latency-bound; NM_GRAPH=0/1 in the
 * environment at nm_mesh_create forces off/on), when a step arrives with the arguments of the
 * step before it (scheme, dt, m_inout, renormalise, rtol, atol, the arrays and h_uniform of
 * `zeeman`) and zeeman->amp is NULL, its kernel launches are captured once into a CUDA graph
 * and replayed with one launch on `stream`; same kernels, same arguments, identical results.
 * The arrays `zeeman` points to are then read at replay time, as the launches would.  The same
 * holds for nm_adjoint_rk4_step[_hext] (key: dt, m_inout, a_inout, u_inout, u_h_inout, renormalise,
 * zeeman). */
nm_status nm_rk_step(nm_mesh *mesh, nm_scheme scheme, double t, double dt, void *m_inout,
                     const nm_zeeman *zeeman, int renormalise, double rtol, double atol,
                     double *err_norm_host, void *stream);

/* a11: right-hand sides of the adjoint-state system Eq. (29) for theta = Ms (cell-wise):
 *   dmdt_out    = f(t, m)                         (may be NULL)
 *   dadt_out    = -(df/dm)^T a                    (nodal 3-vector)
 *   dudt_Ms_out = -(df/dMs)^T a                   (cell scalar, may be NULL)
 * with the explicit transposed operators of reading C7 (two demag convolutions). */
nm_status nm_llg_adjoint_rhs(nm_mesh *mesh, double t, const void *m, const void *a,
                             const nm_zeeman *zeeman, void *dmdt_out, void *dadt_out,
                             void *dudt_Ms_out, void *stream);

/* One RK4 step of size -dt of the augmented system (m, a, u) of Eq. (29), integrating backwards
 * from t to t - dt (reading C8); m is renormalised after the step if renormalise != 0.
 * u_inout is the cell-wise accumulator whose value at t = 0 is grad_Ms of the objective (Eq. 30). */
nm_status nm_adjoint_rk4_step(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                              void *u_inout, const nm_zeeman *zeeman, int renormalise, void *stream);

/* Gradient with respect to a spatially uniform external field h (added to zeeman->h_uniform): the
 * design variable of the field-angle problem, Eqs. (31)-(33).  A uniform field
 * passes through the weak form of Eq. (21) unchanged at every node with (S Ms)_n > 0, so
 *   -(df/dh)^T a = - sum_{n: (S Ms)_n > 0} b_n,   b = g' m x a - alpha g' m x (m x a)
 * (fp64 accumulation in a fixed order; zero when the mesh has no Zeeman term).
 *   nm_llg_adjoint_rhs_hext: dudt_h_out[3] (DEVICE, fp64) = that 3-vector for the given m, a.
 *   nm_adjoint_rk4_step_hext: nm_adjoint_rk4_step that also integrates u_h_inout[3] (DEVICE, fp64)
 *   backwards; with u_h(T) = 0, u_h(0) = dL/dh. */
nm_status nm_llg_adjoint_rhs_hext(nm_mesh *mesh, const void *m, const void *a, double *dudt_h_out,
                                  void *stream);
nm_status nm_adjoint_rk4_step_hext(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                                   void *u_inout, double *u_h_inout, const nm_zeeman *zeeman,
                                   int renormalise, void *stream);

/* The same uniform-field gradient for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no nm_mesh and no workspace are needed, and the call makes no
 * cudaMalloc / cudaFree and calls no allocating library routine.  Its per-block partial sums live in a
 * file-scope device array of libnm.so (192 KB, held by every GPU that loads the library until the process exits),
 * which limits the mesh to NM_NOALLOC_MAX_NODES nodes, (N1+1)(N2+1)(N3+1); more is NM_EINVAL.
 *   device      the GPU the arrays live on (made current by the call); 0 <= device < 64
 *   dtype       precision of m, a, Ms
 *   n_cells     HOST, N1, N2, N3 >= 1 (3-D nodal basis)
 *   m, a        DEVICE nodal 3-vector fields [3][N3+1][N2+1][N1+1]
 *   Ms          DEVICE cell array [N3][N2][N1], or NULL = magnetic everywhere; a node counts if some cell that
 *               contains it has Ms > 0 (reading C3(iii): nodes with (S Ms)_n = 0 see no field)
 *   gamma, alpha  as in nm_mesh_desc
 *   dudt_h_out  DEVICE fp64 [3], overwritten: - sum_{n: (S Ms)_n > 0} b_n,  b = g' m x a - alpha g' m x (m x a),
 *               what nm_llg_adjoint_rhs_hext gives on a mesh with NM_TERM_ZEEMAN (fp64 sums in a fixed order)
 * Enqueues two kernels on `stream`.  All calls on one device share the scratch array: it keeps the last call's
 * partial sums, each call overwrites what it reads (nothing needs clearing), and calls that OVERLAP on the GPU
 * (different streams without an ordering between them) race on it -- order them, or use the mesh entry point.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress); make it outside stream capture. */
#define NM_NOALLOC_MAX_NODES (1ll << 25)
nm_status nm_hext_gradient_noalloc(int device, nm_dtype dtype, const int *n_cells, const void *m, const void *a,
                                   const void *Ms, double gamma, double alpha, double *dudt_h_out, void *stream);

/* Gradients with respect to the cell-wise exchange constant A_c and anisotropy constant Ku_c (design
 * variables beside Ms).  f depends on them through H = -dE/L only, dE linear in
 * both (Eqs. 19-20, 22), so with b as above and bL = b / L (0 at nodes with L_n = 0), K and M the
 * element matrices of Eq. (12):
 *   -(df/dA_c)^T a  = +2 sum_{i,i'} K[i,i'] bL_{c+i} . m_{c+i'}
 *   -(df/dKu_c)^T a = -2 sum_{i,i'} M[i,i'] (bL_{c+i}.k) (m_{c+i'}.k)
 * (zero for a term the mesh does not have).  Outputs are DEVICE cell arrays [N3][N2][N1] of the mesh
 * dtype; either may be NULL.
 *   nm_llg_adjoint_rhs_materials: the two right-hand sides for the given m, a.
 *   nm_adjoint_rk4_step_ex: nm_adjoint_rk4_step that also integrates the accumulators named in
 *   `extra` backwards (any of them NULL = not wanted); with u_X(T) = 0, u_X(0) = dL/dX. */
typedef struct {
    void *u_A, *u_Ku;     /* device cell arrays, mesh dtype, in/out */
    double *u_h;          /* device fp64 [3], in/out (uniform external field, see above) */
    void *u_hn;           /* device nodal 3-vector field, mesh dtype, in/out: gradient with respect to a
                             time-constant NODAL external field (nm_llg_adjoint_rhs_hnodal) */
} nm_adjoint_extra;

/* -(df/dh)^T a for a nodal external field h(n) entering through the weak form of Eq. (21) (
 * SURVEY.md 8(f) row 2 lists H^ext among the design variables): with b = (df/dH)^T a,
 *   dudt_hn_out = Z(b / L),  Z h = -mu0 sum_c Ms_c sum_i' M_{i,i'} h_{c+i'}  (the Zeeman variation, symmetric),
 * a nodal 3-vector field of the mesh dtype; zero without NM_TERM_ZEEMAN and at nodes with (S Ms)_n = 0 all round.
 * Summed over the nodes it equals nm_llg_adjoint_rhs_hext.  Uses the mesh's adjoint scratch. */
nm_status nm_llg_adjoint_rhs_hnodal(nm_mesh *mesh, const void *m, const void *a, void *dudt_hn_out, void *stream);
nm_status nm_llg_adjoint_rhs_materials(nm_mesh *mesh, const void *m, const void *a, void *dudt_A_out,
                                       void *dudt_Ku_out, void *stream);
nm_status nm_adjoint_rk4_step_ex(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                                 void *u_inout, const nm_adjoint_extra *extra, const nm_zeeman *zeeman,
                                 int renormalise, void *stream);

/* Objectives at several times T_i ("adding appropriate terms depending on m(T_i)"):
 * when the backward integration of Eq. (29) arrives at T_i the adjoint variable takes the jump
 *   a_inout <- a_inout + scale * dLdm     (device nodal 3-vectors of the mesh dtype),
 * dLdm = grad_m L_i(m(T_i)) from the caller.  a_inout and dLdm must not overlap. */
nm_status nm_adjoint_add_objective(nm_mesh *mesh, void *a_inout, const void *dLdm, double scale,
                                   void *stream);

/* Debug / test getters (not hot path).  Copy the real-space demag tensor N[6][N3][N2][N1]
 * (components xx,yy,zz,xy,xz,yz; non-negative cell offsets; fp64) to a HOST buffer, and the
 * cell-wise demag field [3][N3][N2][N1] of the last nm_heff/nm_llg_rhs call (mesh dtype) to a
 * DEVICE buffer. */
nm_status nm_debug_get_tensor(nm_mesh *mesh, double *N_host);
nm_status nm_debug_get_cell_field(nm_mesh *mesh, void *Hc_out, void *stream);

/* Number of kernel launches this library has issued on this mesh since create (for bench). */
long long nm_launch_count(const nm_mesh *mesh);

/* Which demag kernels serve this mesh (tests check that a grid takes the path they mean to cover):
 * 0 no demag term or general-size kernels, 1 register-FFT fast path (every N_d = 16 * 2^k),
 * 2 fast path on the mesh zero-extended to the next sizes 16 * 2^k. */
int nm_debug_demag_path(const nm_mesh *mesh);

/* Per-kernel timing for the roofline line of bench.py.  Between
 * nm_profile_begin and nm_profile_end every kernel launch on this mesh is bracketed by a pair of
 * CUDA events on the launching stream (at most 4096 launches are recorded; later ones are counted
 * by nm_launch_count and nm_profile_dropped, so a caller can tell that its shares are incomplete).
 * nm_profile_end synchronises `stream` and writes, for each of the nm_profile_class_count() kernel classes, the summed device time in milliseconds and the number
 * of recorded launches to the two HOST arrays (each of nm_profile_class_count() entries).
 * nm_profile_class_name(i) names class i ("x_fwd", "y_fwd", "mid", "y_inv", "x_inv", "node",
 * "adj_cell", "lincomb", "other", "node_rk", "node_adj": the node pass is split by what its epilogue
 * moves -- H or f alone, a Runge-Kutta stage, an adjoint pass). */
long long nm_profile_dropped(const nm_mesh *mesh); /* launches since nm_profile_begin that were not timed */
int nm_profile_class_count(void);
const char *nm_profile_class_name(int cls);
nm_status nm_profile_begin(nm_mesh *mesh);
nm_status nm_profile_end(nm_mesh *mesh, void *stream, double *ms_host, long long *count_host);

#ifdef __cplusplus
}
#endif
#endif /* NM_H */
