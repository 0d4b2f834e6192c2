// Internal definitions shared by the translation units of libnm.so (not part of the ABI).
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>
#include <string>

#include "../../include/nm.h"

#define NM_MAX_STAGES 20
#define NM_HEXT_BLOCKS 1024
#define NM_PROF_MAX 4096

// kernel classes reported by nm_profile_end (order = NM_PROF_* of include/nm.h)
enum NmKernelClass {
    NM_K_X_FWD = 0, NM_K_Y_FWD, NM_K_MID, NM_K_Y_INV, NM_K_X_INV, NM_K_NODE, NM_K_ADJ_CELL,
    NM_K_LINCOMB, NM_K_OTHER, NM_K_NODE_RK, NM_K_NODE_ADJ, NM_K_COUNT
};
// the node pass by what its epilogue moves: H / f alone ("node"), a Runge-Kutta stage that also reads
// the start-of-step state and earlier derivatives and writes the derivative and the next stage state
// ("node_rk"), the two adjoint passes ("node_adj"); mode = NmLocalMode of nm_local.cuh
inline int nm_node_class(int mode) { return mode <= 1 ? NM_K_NODE : mode == 2 ? NM_K_NODE_RK : NM_K_NODE_ADJ; }
#define NM_MU0 (4.0e-7 * 3.14159265358979323846264338327950288)

// ------------------------------------------------------------------------------------------------
// FFT plan for one axis: complex transform of length L as a product of radix-{8,4,2,3} stages.
// Forward = decimation in frequency (natural order in, digit-reversed out), inverse = the
// adjoint stages in reverse order (digit-reversed in, natural out), so a convolution needs no
// reordering pass: the spectrum lives in digit-reversed ("position") order everywhere and
// kmap[pos] gives the frequency index of a position, pos[k] its inverse.
struct NmFftPlan {
    int L;
    int n_stages;
    int radix[NM_MAX_STAGES];
};

template <typename T> struct NmVec2;
template <> struct NmVec2<float> { typedef float2 type; };
template <> struct NmVec2<double> { typedef double2 type; };

// Geometry and workspace pointers handed to kernels by value.
struct NmGeom {
    int N1, N2, N3;    // cells
    int n1, n2, n3;    // stored node extents: cells + 1, or 1 along an axis the basis does not vary in
    int ys, zs;        // element stride from a node to its +y / +z neighbour (n1, n1 n2), or 0 along a reduced
                       // axis: the neighbour is the node itself, i.e. the state is uniform along that axis and
                       // the 3-D operators applied to it are the reduced scheme (Eqs. 23-24)
    int P1, P2, P3;    // padded FFT lengths (2 N_d, or 1 if N_d == 1)
    int C1;            // complex outputs of the x transform: N1 + 1 (or 1)
    int C1p;           // row pitch of spectrum buffers, complex elements
    int K2, K3;        // folded frequency counts along y, z: N_d + 1 (or 1)
    int Lx;            // complex length of the packed x transform: N1 (P1/2)
    long long cells, nodes;
};

// Opaque copy of a CUtensorMap (128 bytes, 64-byte aligned) so that this header does not need cuda.h
struct alignas(64) NmTensorMap {
    unsigned char bytes[128];
};

// Fast demag path (nm_demag_fast.cu): sizes 16 M_d per axis, blocked spectrum layouts.
struct NmFast {
    bool on;
    int M1, M2, M3;    // F_d / 16
    int F1, F2, F3;    // transform extents: F_d = N_d, or the next fast size above N_d (embedded mesh)
    bool embed;        // some F_d > N_d: the mesh is zero-extended to the fast size (fp32 pipelined kernels only)
    int Wx;            // warps per CTA of the x passes
    int NKT;           // k1 tiles of 8 columns
    int Kzp;           // pitch of the |kz| axis of the tensor
    int kt_chunk;      // k1 tiles per y/z/y launch group (0 = all)
    bool pipe;         // use the persistent TMA-pipelined kernels (nm_demag_pipe.cu) where they apply
    bool tmapB_ok;     // tmapB describes bufB (fp32, N2 = 256)
    NmTensorMap tmapB; // 4-D tiled view of bufB for the pipelined y passes
    void *Tn;          // tensor [NKT][N2+1][8][6][Kzp] (real)
    void *wPx;         // exp(-2 pi i q / P1), q < P1
};

// One cached time step: the arguments that fix its launch sequence, and the instantiated graph
// (null until the same arguments arrive a second time in a row).
struct NmStepKey {
    int kind, renorm, has_z, pad;   // no implicit padding: keys are compared with memcmp
    double dt, rtol, atol, hu[3];
    const void *p[7], *hs, *hp;
    unsigned long long epoch;
};
struct NmStepGraph {
    bool seen;
    NmStepKey key;
    cudaGraphExec_t exec;
    long long launches;                // kernels in the graph
};
enum { NM_GRAPH_RK4 = 0, NM_GRAPH_DOPRI5, NM_GRAPH_ADJ_RK4, NM_GRAPH_SLOTS };

struct nm_mesh {
    nm_mesh_desc desc;
    NmGeom g;
    NmFast fast;
    bool f64;
    size_t esz;        // sizeof(real)
    int sm_count;
    long long launches;
    // FFT plans
    NmFftPlan plan_x, plan_y, plan_z;
    // device pointers inside the caller's workspace
    char *ws;
    size_t ws_bytes;
    void *Ms, *A, *Ku;      // cell scalars (real)
    void *sMs;              // nodal S Ms (real)
    double *Nreal;          // [6][N3][N2][N1] fp64 real-space tensor
    void *Nhat;             // [6][K3][K2][C1p] real spectrum, scaled by 1/(P1 P2 P3)
    void *tw_x, *tw_x2, *tw_y, *tw_z;   // complex twiddle tables
    int *kmap_x, *pos_x, *kmap_y, *pos_y, *kmap_z, *pos_z;
    void *bufA, *bufB;      // spectrum buffers (complex)
    void *Hc1, *Hc2;        // cell demag fields [3][cells]
    void *Q, *W;            // adjoint scratch: nodal vector, nodal scalar
    void *Zs;               // weak-form nodal Zeeman field of the current stage (nodal vector), or null
    void *Dmi, *Kcub;       // cell scalars of NM_TERM_DMI / NM_TERM_CUBIC (real), or null
    void *Xs;               // field of those terms at the current stage (nodal vector), or null
    void *K[7];             // RK stage derivatives (nodal vectors)
    void *Y[2];             // RK stage states
    void *Uc[2];            // cell scalars (adjoint RK)
    double *hpart;          // partial sums of the uniform-field gradient [3][NM_HEXT_BLOCKS]
    double *partials;       // reduction scratch [node blocks + 1]
    int n_partials;         // capacity
    int last_partials;      // partial sums the last node-kernel launch wrote
    // materials given as scalars at create (enables the separable node kernel)
    bool uni_A, uni_Ku, uni_Ms;
    bool hc1_valid;
    int dbg_node_path;      // NM_NODE_PATH at create: 0 automatic, 1 27-point kernel, 2 k_node_sep, 3 column kernel fed by cp.async (tests)
    // per-launch timing (nm_profile_begin / nm_profile_end)
    bool prof_on;
    int prof_n;
    long long prof_dropped; // launches since nm_profile_begin that found the event table full (not timed)
    int prof_cls[NM_PROF_MAX];
    cudaEvent_t prof_ev[NM_PROF_MAX][2];
    int prof_ev_made;       // events created so far (created lazily, destroyed with the mesh)
    // Replay of whole time steps as CUDA graphs (launch-latency-bound meshes; nm_api.cu)
    bool graph_on;
    cudaStream_t cap_stream;           // capture vehicle, created lazily (nothing ever runs on it)
    unsigned long long graph_epoch;    // bumped by whatever changes the launch sequence (nm_mesh_set_Ms)
    NmStepGraph step_graph[NM_GRAPH_SLOTS];
};

// 2^(D-3) for a nodal basis that varies in D axes (1 on the 3-D basis).  The kernels reach a reduced basis through
// zero node strides along the reduced axes, which counts every vertex of a cell 2^(3-D) times and keeps the 3-D
// lumped mass V / 8: the cell-wise gradients of the adjoint entry points take this factor once (a node kernel sees
// only its own half of each reduced axis, (1/3 + 1/6) of the mass row, which cancels against V / 8 vs V / 2^D).
inline double nm_red_scale(const nm_mesh *m)
{
    const int D = m->desc.basis == 0 ? 3 : m->desc.basis;
    return D >= 3 ? 1.0 : (D == 2 ? 0.5 : 0.25);
}

// Brackets one kernel launch with an event pair when profiling is on, and counts it.
struct NmLaunchScope {
    nm_mesh *m;
    cudaStream_t st;
    int slot;
    NmLaunchScope(nm_mesh *mesh, int cls, cudaStream_t stream) : m(mesh), st(stream), slot(-1)
    {
        m->launches++;
        if (m->prof_on && m->prof_n >= NM_PROF_MAX) m->prof_dropped++;
        if (m->prof_on && m->prof_n < NM_PROF_MAX) {
            slot = m->prof_n++;
            if (slot >= m->prof_ev_made) {
                cudaEventCreate(&m->prof_ev[slot][0]);
                cudaEventCreate(&m->prof_ev[slot][1]);
                m->prof_ev_made = slot + 1;
            }
            m->prof_cls[slot] = cls;
            cudaEventRecord(m->prof_ev[slot][0], st);
        }
    }
    ~NmLaunchScope()
    {
        if (slot >= 0) cudaEventRecord(m->prof_ev[slot][1], st);
    }
};

void nm_set_error(const char *fmt, ...);

#define NM_CUDA_TRY(expr)                                                                       \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            nm_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__,     \
                         __LINE__);                                                             \
            return NM_ECUDA;                                                                    \
        }                                                                                       \
    } while (0)

#define NM_TRY(expr)                                                                            \
    do {                                                                                        \
        nm_status s_ = (expr);                                                                  \
        if (s_ != NM_OK) return s_;                                                             \
    } while (0)

// nm_tensor.cu
nm_status nm_build_tensor(nm_mesh *mesh, cudaStream_t st);
// nm_demag.cu
template <typename T>
nm_status nm_demag_conv(nm_mesh *mesh, const T *field_nodes, T *Hc_out, cudaStream_t st);
// nm_demag_fast.cu
void nm_fast_plan(const nm_mesh_desc *d, const NmGeom &g, NmFast *f);
size_t nm_fast_tensor_elems(const NmGeom &g, const NmFast &f);
size_t nm_fast_bufA_elems(const NmGeom &g, const NmFast &f);
size_t nm_fast_bufB_elems(const NmGeom &g, const NmFast &f);
nm_status nm_fast_store_tensor(nm_mesh *mesh, const double *octant, double scale, cudaStream_t st);
template <typename T>
nm_status nm_demag_conv_fast(nm_mesh *mesh, const T *field_nodes, T *Hc_out, cudaStream_t st);
// nm_demag_pipe.cu
bool nm_pipe_mid_ok(const nm_mesh *mesh);
nm_status nm_pipe_mid(nm_mesh *mesh, int kt0, int nkt, cudaStream_t st);
nm_status nm_pipe_setup(nm_mesh *mesh);      // after the workspace is carved
bool nm_pipe_y_ok(const nm_mesh *mesh);
nm_status nm_pipe_y(nm_mesh *mesh, bool inverse, int kt0, int nkt, cudaStream_t st);
bool nm_pipe_x_ok(const nm_mesh *mesh);
template <typename T> nm_status nm_pipe_x(nm_mesh *mesh, bool inverse, const T *fld, T *Hc, cudaStream_t st);
// nm_local.cu
nm_status nm_compute_sMs(nm_mesh *mesh, cudaStream_t st);

extern "C" int nm_newell_near_box(const int *box, const double *dx, double *out, int n_threads);
