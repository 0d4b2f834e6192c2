// C-ABI entry points of libnm.so (include/nm.h): mesh setup, field / right-hand-side evaluation,
// Runge-Kutta steps and the adjoint right-hand side.  Host orchestration only: every step of the
// path runs in the kernels of nm_local.cu and nm_demag.cu.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "nm_internal.h"
#include "nm_local.cuh"

// ---- errors ------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

void nm_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *nm_last_error(void) { return g_err; }

namespace {

// ---- geometry, FFT plans -----------------------------------------------------------------------
bool smooth7(int n)          // 2^a 3^b 5^c 7^d: the radices of nm_fft.cuh
{
    for (int r = 2; r <= 7; r += (r == 2 ? 1 : 2))
        while (n % r == 0) n /= r;
    return n == 1;
}

void make_plan(int L, NmFftPlan *p)
{
    p->L = L;
    p->n_stages = 0;
    int n = L;
    // odd factors first (largest blocks), then 8s, then what is left of the power of two
    while (n % 7 == 0) { p->radix[p->n_stages++] = 7; n /= 7; }
    while (n % 5 == 0) { p->radix[p->n_stages++] = 5; n /= 5; }
    while (n % 3 == 0) { p->radix[p->n_stages++] = 3; n /= 3; }
    while (n % 8 == 0) { p->radix[p->n_stages++] = 8; n /= 8; }
    if (n % 4 == 0) { p->radix[p->n_stages++] = 4; n /= 4; }
    if (n % 2 == 0) { p->radix[p->n_stages++] = 2; n /= 2; }
}

// Position <-> frequency of the decimation-in-frequency stages (nm_fft.cuh): a stage with block
// length n and radix R leaves the outputs k = t (mod R) in sub-block t.
void make_maps(const NmFftPlan &p, std::vector<int> &kmap, std::vector<int> &pos)
{
    kmap.assign(p.L, 0);
    pos.assign(p.L, 0);
    for (int q = 0; q < p.L; ++q) {
        int rem = q, m = p.L, k = 0, w = 1;
        for (int s = 0; s < p.n_stages; ++s) {
            m /= p.radix[s];
            const int t = rem / m;
            rem -= t * m;
            k += t * w;
            w *= p.radix[s];
        }
        kmap[q] = k;
        pos[k] = q;
    }
}

void make_geom(const nm_mesh_desc *d, NmGeom *g);

nm_status validate(const nm_mesh_desc *d)
{
    if (!d) { nm_set_error("desc is NULL"); return NM_EINVAL; }
    for (int i = 0; i < 3; ++i) {
        if (d->n_cells[i] < 1) { nm_set_error("n_cells[%d] = %d < 1", i, d->n_cells[i]); return NM_EINVAL; }
        if (!(d->cell_size[i] > 0)) { nm_set_error("cell_size[%d] must be > 0", i); return NM_EINVAL; }
    }
    if (d->dtype != NM_F32 && d->dtype != NM_F64) { nm_set_error("bad dtype"); return NM_EINVAL; }
    if (d->basis < 0 || d->basis > 3) { nm_set_error("basis = %d is not 0, 1, 2 or 3", d->basis); return NM_EINVAL; }
    if ((d->basis == 2 && d->n_cells[2] != 1) || (d->basis == 1 && (d->n_cells[1] != 1 || d->n_cells[2] != 1))) {
        nm_set_error("a %d-D basis needs one cell along the reduced axes (n_cells = %d x %d x %d)", d->basis,
                     d->n_cells[0], d->n_cells[1], d->n_cells[2]);
        return NM_EINVAL;
    }
    if (d->terms == 0 || (d->terms & ~127u)) { nm_set_error("terms = %u is not a combination of NM_TERM_*", d->terms); return NM_EINVAL; }
    if (d->terms & (NM_TERM_DMI | NM_TERM_CUBIC | NM_TERM_RKKY)) {
        if (d->basis != 0 && d->basis != 3) {
            nm_set_error("NM_TERM_DMI / NM_TERM_CUBIC / NM_TERM_RKKY are written for the 3-D basis (basis = %d)", d->basis);
            return NM_EUNSUPPORTED;
        }
        if (d->terms & NM_TERM_RKKY) {
            const int za = d->rkky_planes[0], zb = d->rkky_planes[1];
            if (za == zb || za < 0 || zb < 0 || za > d->n_cells[2] || zb > d->n_cells[2]) {
                nm_set_error("rkky_planes = (%d, %d) must be two different node planes in [0, N3]", za, zb);
                return NM_EINVAL;
            }
        }
        if ((d->terms & NM_TERM_DMI) && (d->dmi_kind < 0 || d->dmi_kind > 1 || d->dmi_normal < 0 || d->dmi_normal > 2)) {
            nm_set_error("dmi_kind = %d / dmi_normal = %d out of range", d->dmi_kind, d->dmi_normal);
            return NM_EINVAL;
        }
        if (d->terms & NM_TERM_CUBIC) {
            const double *c = d->cubic_axes;
            for (int q = 0; q < 3; ++q)
                for (int r = q; r < 3; ++r) {
                    const double dot = c[3 * q] * c[3 * r] + c[3 * q + 1] * c[3 * r + 1] + c[3 * q + 2] * c[3 * r + 2];
                    if (std::fabs(dot - (q == r ? 1.0 : 0.0)) > 1e-9) {
                        nm_set_error("cubic_axes must be three orthonormal rows");
                        return NM_EINVAL;
                    }
                }
        }
    }
    if (!(d->gamma == d->gamma) || !(d->alpha == d->alpha)) { nm_set_error("gamma / alpha is NaN"); return NM_EINVAL; }
    if (d->terms & NM_TERM_ANISO) {
        const double *k = d->ku_axis;
        const double n2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
        if (std::fabs(n2 - 1.0) > 1e-9) { nm_set_error("ku_axis must be a unit vector"); return NM_EINVAL; }
    }
    if (d->terms & NM_TERM_DEMAG) {
        // a mesh the zero-extended fast path serves needs no factorisation of its own
        NmGeom ge;
        NmFast fe;
        make_geom(d, &ge);
        nm_fast_plan(d, ge, &fe);
        const bool embedded = fe.on && fe.embed && !getenv("NM_DEMAG_PATH") && !getenv("NM_PIPE");
        for (int i = 0; i < 3; ++i)
            if (!embedded && d->n_cells[i] > 1 && !smooth7(d->n_cells[i])) {
                nm_set_error("n_cells[%d] = %d is not of the form 2^a 3^b 5^c 7^d (demag FFT radices)", i, d->n_cells[i]);
                return NM_EUNSUPPORTED;
            }
        const size_t cx = d->dtype == NM_F64 ? 16 : 8;
        if ((size_t)12 * d->n_cells[0] * cx > 200 * 1024) {
            nm_set_error("n_cells[0] = %d too long for the x pass", d->n_cells[0]);
            return NM_EUNSUPPORTED;
        }
    }
    return NM_OK;
}

void make_geom(const nm_mesh_desc *d, NmGeom *g)
{
    g->N1 = d->n_cells[0]; g->N2 = d->n_cells[1]; g->N3 = d->n_cells[2];
    const int basis = d->basis == 0 ? 3 : d->basis;
    g->n1 = g->N1 + 1;
    g->n2 = basis >= 2 ? g->N2 + 1 : 1;
    g->n3 = basis >= 3 ? g->N3 + 1 : 1;
    g->ys = basis >= 2 ? g->n1 : 0;
    g->zs = basis >= 3 ? g->n1 * g->n2 : 0;
    g->P1 = g->N1 > 1 ? 2 * g->N1 : 1;
    g->P2 = g->N2 > 1 ? 2 * g->N2 : 1;
    g->P3 = g->N3 > 1 ? 2 * g->N3 : 1;
    g->C1 = g->N1 > 1 ? g->N1 + 1 : 1;
    g->C1p = (g->C1 + 3) & ~3;
    g->K2 = g->N2 > 1 ? g->N2 + 1 : 1;
    g->K3 = g->N3 > 1 ? g->N3 + 1 : 1;
    g->Lx = g->N1;
    g->cells = (long long)g->N1 * g->N2 * g->N3;
    g->nodes = (long long)g->n1 * g->n2 * g->n3;
}

// Bump allocator over the caller's workspace; with base == nullptr it only measures.
struct Carver {
    char *base;
    size_t off;
    void *take(size_t bytes)
    {
        off = (off + 255) & ~(size_t)255;
        void *p = base ? base + off : nullptr;
        off += bytes;
        return p;
    }
};

size_t carve(nm_mesh *m, char *base)
{
    const NmGeom &g = m->g;
    const size_t e = m->esz, cx = 2 * m->esz;
    const bool demag = (m->desc.terms & NM_TERM_DEMAG) != 0;
    Carver c{base, 0};
    m->Ms = c.take(g.cells * e);
    m->A = c.take(g.cells * e);
    m->Ku = c.take(g.cells * e);
    m->sMs = c.take(g.nodes * e);
    m->n_partials = nm_node_blocks(g);
    m->partials = (double *)c.take(((size_t)m->n_partials + 1) * sizeof(double));
    m->hpart = (double *)c.take((size_t)3 * NM_HEXT_BLOCKS * sizeof(double));
    // Runge-Kutta / adjoint scratch; doubles as fp64 scratch of the tensor setup
    const size_t vec = (size_t)3 * g.nodes * e;
    // every stage array starts on a 256-byte boundary (3 nodes e is odd-sized): the bulk-copy feeds of the x pass
    // and of the node kernel need 16-byte aligned nodal arrays, and a stage state is the field of the next stage
    const size_t vecp = (vec + 255) & ~(size_t)255;
    size_t rk = 9 * vecp;
    if (demag) {
        const size_t need = (size_t)2 * 6 * g.C1 * g.K2 * g.K3 * sizeof(double);
        if (need > rk) rk = need;
    }
    char *r = (char *)c.take(rk);
    for (int i = 0; i < 7; ++i) m->K[i] = r ? r + i * vecp : nullptr;
    for (int i = 0; i < 2; ++i) m->Y[i] = r ? r + (7 + i) * vecp : nullptr;
    m->Q = c.take(vec);
    m->W = c.take(g.nodes * e);
    m->Uc[0] = c.take(g.cells * e);
    m->Uc[1] = c.take(g.cells * e);
    m->Zs = (m->desc.terms & NM_TERM_ZEEMAN) ? c.take(vec) : nullptr;
    m->Dmi = (m->desc.terms & NM_TERM_DMI) ? c.take(g.cells * e) : nullptr;
    m->Kcub = (m->desc.terms & NM_TERM_CUBIC) ? c.take(g.cells * e) : nullptr;
    m->Xs = (m->desc.terms & (NM_TERM_DMI | NM_TERM_CUBIC | NM_TERM_RKKY)) ? c.take(vec) : nullptr;
    m->Hc1 = m->Hc2 = nullptr;
    m->Nreal = nullptr;
    m->fast.Tn = m->fast.wPx = nullptr;
    m->Nhat = m->tw_x = m->tw_x2 = m->tw_y = m->tw_z = m->bufA = m->bufB = nullptr;
    m->kmap_x = m->pos_x = m->kmap_y = m->pos_y = m->kmap_z = m->pos_z = nullptr;
    if (demag) {
        m->Hc1 = c.take(3 * g.cells * e);
        m->Hc2 = c.take(3 * g.cells * e);
        m->Nreal = (double *)c.take(6 * g.cells * sizeof(double));
        if (m->fast.on) {
            m->fast.Tn = c.take(nm_fast_tensor_elems(g, m->fast) * e);
            m->fast.wPx = c.take((size_t)g.P1 * cx);
        } else {
            m->Nhat = c.take((size_t)6 * g.K3 * g.K2 * g.C1p * e);
        }
        m->tw_x = c.take((size_t)g.Lx * cx);
        m->tw_x2 = c.take((size_t)g.C1 * cx);
        m->tw_y = c.take((size_t)g.P2 * cx);
        m->tw_z = c.take((size_t)g.P3 * cx);
        m->kmap_x = (int *)c.take(g.Lx * sizeof(int));
        m->pos_x = (int *)c.take(g.Lx * sizeof(int));
        m->kmap_y = (int *)c.take(g.P2 * sizeof(int));
        m->pos_y = (int *)c.take(g.P2 * sizeof(int));
        m->kmap_z = (int *)c.take(g.P3 * sizeof(int));
        m->pos_z = (int *)c.take(g.P3 * sizeof(int));
        if (m->fast.on) {
            m->bufA = c.take(nm_fast_bufA_elems(g, m->fast) * cx);
            m->bufB = c.take(nm_fast_bufB_elems(g, m->fast) * cx);
        } else {
            m->bufA = c.take((size_t)3 * g.N3 * g.N2 * g.C1p * cx);
            if (g.N3 > 1) m->bufB = c.take((size_t)3 * g.N3 * g.P2 * g.C1p * cx);
        }
    }
    return (c.off + 255) & ~(size_t)255;
}

void init_host(nm_mesh *m, const nm_mesh_desc *d)
{
    m->desc = *d;
    make_geom(d, &m->g);
    m->f64 = d->dtype == NM_F64;
    m->esz = m->f64 ? 8 : 4;
    m->launches = 0;
    m->last_partials = 0;
    m->uni_A = d->A == nullptr;
    m->uni_Ku = d->Ku == nullptr;
    m->uni_Ms = d->Ms == nullptr;
    m->hc1_valid = false;
    m->prof_on = false;
    m->prof_n = 0;
    m->prof_dropped = 0;
    m->prof_ev_made = 0;
    {
        // whole steps of small meshes are launch-latency-bound: replay them as graphs (NM_GRAPH=0 / 1
        // forces the choice)
        const char *ge = getenv("NM_GRAPH");
        m->graph_on = ge ? atoi(ge) != 0 : m->g.cells <= (1LL << 21);
        m->cap_stream = nullptr;
        m->graph_epoch = 0;
        memset(m->step_graph, 0, sizeof(m->step_graph));
    }
    {
        // test switch, read here once (never on the evaluation path): NM_NODE_PATH = "generic" forces the
        // 27-point node kernel, "sep" k_node_sep
        const char *env = getenv("NM_NODE_PATH");
        m->dbg_node_path = env && strcmp(env, "generic") == 0 ? 1 : env && strcmp(env, "sep") == 0 ? 2 :
                           env && strcmp(env, "ring") == 0 ? 3 : 0;     // "ring": the cp.async form of the column kernel
    }
    nm_fast_plan(d, m->g, &m->fast);
    {
        const char *env = getenv("NM_DEMAG_PATH");      // "generic" forces the general-size kernels
        if (env && strcmp(env, "generic") == 0) m->fast.on = false;
        const char *ch = getenv("NM_KT_CHUNK");
        m->fast.kt_chunk = ch ? atoi(ch) : 0;
        const char *pp = getenv("NM_PIPE");              // "0" forces the non-pipelined fast kernels
        m->fast.pipe = !(pp && strcmp(pp, "0") == 0);
        if (m->fast.embed && !m->fast.pipe) m->fast.on = false;   // embedded meshes exist in the pipelined kernels only
        if (!m->fast.on) m->fast.embed = false;
    }
    if (m->fast.on && m->fast.embed) {      // spectral extents follow the transform sizes
        NmGeom &g = m->g;
        const NmFast &f = m->fast;
        g.P1 = 2 * f.F1; g.P2 = 2 * f.F2; g.P3 = 2 * f.F3;
        g.C1 = f.F1 + 1;
        g.C1p = (g.C1 + 3) & ~3;
        g.K2 = f.F2 + 1;
        g.K3 = f.F3 + 1;
        g.Lx = f.F1;
    }
    make_plan(m->g.Lx, &m->plan_x);
    make_plan(m->g.P2, &m->plan_y);
    make_plan(m->g.P3, &m->plan_z);
}

template <typename T> __global__ void k_fill(T *p, long long n, T v)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

template <typename T>
nm_status set_material(nm_mesh *m, void *dst, const void *src, double scalar, cudaStream_t st)
{
    const long long n = m->g.cells;
    if (src) {
        NM_CUDA_TRY(cudaMemcpyAsync(dst, src, n * sizeof(T), cudaMemcpyDeviceToDevice, st));
    } else {
        {
            NmLaunchScope sc(m, NM_K_OTHER, st);
            k_fill<T><<<(unsigned)((n + 255) / 256), 256, 0, st>>>((T *)dst, n, (T)scalar);
        }
        NM_CUDA_TRY(cudaGetLastError());
    }
    return NM_OK;
}

// exp(-2 pi i q / L), q = 0..count-1, evaluated in fp64 and rounded to the mesh dtype
template <typename T>
nm_status upload_twiddles(void *dst, int L, int count, cudaStream_t st)
{
    typedef typename NmVec2<T>::type V;
    std::vector<V> h(count);
    for (int q = 0; q < count; ++q) {
        // exact octant reduction keeps cos/sin at multiples of pi/2 exact
        const double x = 2.0 * (double)q / (double)L;   // angle / pi
        double c, s;
        const long long q8 = (long long)q * 8;
        if (q8 % L == 0 && (q8 / L) % 2 == 0) {
            const int oct = (int)((q8 / L) / 2) & 3;     // multiples of pi/2
            const double cc[4] = {1, 0, -1, 0}, ss[4] = {0, 1, 0, -1};
            c = cc[oct]; s = ss[oct];
        } else {
            c = std::cos(M_PI * x);
            s = std::sin(M_PI * x);
        }
        h[q].x = (T)c;
        h[q].y = (T)(-s);
    }
    NM_CUDA_TRY(cudaMemcpyAsync(dst, h.data(), count * sizeof(V), cudaMemcpyHostToDevice, st));
    NM_CUDA_TRY(cudaStreamSynchronize(st));
    return NM_OK;
}

nm_status upload_ints(int *dst, const std::vector<int> &v, cudaStream_t st)
{
    NM_CUDA_TRY(cudaMemcpyAsync(dst, v.data(), v.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    NM_CUDA_TRY(cudaStreamSynchronize(st));
    return NM_OK;
}

template <typename T> nm_status setup_tables(nm_mesh *m, cudaStream_t st)
{
    const NmGeom &g = m->g;
    NM_TRY(upload_twiddles<T>(m->tw_x, g.Lx, g.Lx, st));
    NM_TRY(upload_twiddles<T>(m->tw_x2, g.P1, g.C1, st));
    NM_TRY(upload_twiddles<T>(m->tw_y, g.P2, g.P2, st));
    NM_TRY(upload_twiddles<T>(m->tw_z, g.P3, g.P3, st));
    if (m->fast.on) NM_TRY(upload_twiddles<T>(m->fast.wPx, g.P1, g.P1, st));
    std::vector<int> km, ps;
    make_maps(m->plan_x, km, ps);
    NM_TRY(upload_ints(m->kmap_x, km, st));
    NM_TRY(upload_ints(m->pos_x, ps, st));
    make_maps(m->plan_y, km, ps);
    NM_TRY(upload_ints(m->kmap_y, km, st));
    NM_TRY(upload_ints(m->pos_y, ps, st));
    make_maps(m->plan_z, km, ps);
    NM_TRY(upload_ints(m->kmap_z, km, st));
    NM_TRY(upload_ints(m->pos_z, ps, st));
    return NM_OK;
}

} // namespace

// ---- mesh life cycle ---------------------------------------------------------------------------
extern "C" nm_status nm_mesh_query_workspace(const nm_mesh_desc *desc, size_t *bytes_out)
{
    NM_TRY(validate(desc));
    if (!bytes_out) { nm_set_error("bytes_out is NULL"); return NM_EINVAL; }
    nm_mesh tmp;
    init_host(&tmp, desc);
    *bytes_out = carve(&tmp, nullptr);
    return NM_OK;
}

extern "C" nm_status nm_mesh_set_Ms(nm_mesh *mesh, const void *Ms, void *stream)
{
    if (!mesh || !Ms) { nm_set_error("NULL argument"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    NM_CUDA_TRY(cudaSetDevice(mesh->desc.device));
    NM_CUDA_TRY(cudaMemcpyAsync(mesh->Ms, Ms, mesh->g.cells * mesh->esz, cudaMemcpyDeviceToDevice, st));
    mesh->hc1_valid = false;
    mesh->uni_Ms = false;
    mesh->graph_epoch++;
    return nm_compute_sMs(mesh, st);
}

extern "C" nm_status nm_mesh_create(nm_mesh **out, const nm_mesh_desc *desc, void *workspace, size_t bytes)
{
    if (!out) { nm_set_error("out is NULL"); return NM_EINVAL; }
    *out = nullptr;
    NM_TRY(validate(desc));
    if (!workspace || ((uintptr_t)workspace & 255)) {
        nm_set_error("workspace must be a 256-byte aligned device pointer");
        return NM_EINVAL;
    }
    nm_mesh *m = new (std::nothrow) nm_mesh;
    if (!m) { nm_set_error("host allocation failed"); return NM_ENOMEM; }
    init_host(m, desc);
    const size_t need = carve(m, (char *)workspace);
    if (bytes < need) {
        nm_set_error("workspace of %zu bytes is smaller than the %zu required", bytes, need);
        delete m;
        return NM_ENOMEM;
    }
    m->ws = (char *)workspace;
    m->ws_bytes = bytes;
    nm_status s = NM_OK;
    cudaStream_t st = 0;
    do {
        cudaError_t e = cudaSetDevice(desc->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, desc->device);
        if (e == cudaSuccess) e = cudaMemsetAsync(workspace, 0, need, st);
        if (e != cudaSuccess) {
            nm_set_error("device setup failed: %s", cudaGetErrorString(e));
            s = NM_ECUDA;
            break;
        }
        if (m->f64) {
            if ((s = set_material<double>(m, m->Ms, desc->Ms, desc->Ms_scalar, st)) != NM_OK) break;
            if ((s = set_material<double>(m, m->A, desc->A, desc->A_scalar, st)) != NM_OK) break;
            if ((s = set_material<double>(m, m->Ku, desc->Ku, desc->Ku_scalar, st)) != NM_OK) break;
            if (m->Dmi && (s = set_material<double>(m, m->Dmi, desc->D, desc->D_scalar, st)) != NM_OK) break;
            if (m->Kcub && (s = set_material<double>(m, m->Kcub, desc->Kc, desc->Kc_scalar, st)) != NM_OK) break;
        } else {
            if ((s = set_material<float>(m, m->Ms, desc->Ms, desc->Ms_scalar, st)) != NM_OK) break;
            if ((s = set_material<float>(m, m->A, desc->A, desc->A_scalar, st)) != NM_OK) break;
            if ((s = set_material<float>(m, m->Ku, desc->Ku, desc->Ku_scalar, st)) != NM_OK) break;
            if (m->Dmi && (s = set_material<float>(m, m->Dmi, desc->D, desc->D_scalar, st)) != NM_OK) break;
            if (m->Kcub && (s = set_material<float>(m, m->Kcub, desc->Kc, desc->Kc_scalar, st)) != NM_OK) break;
        }
        if ((s = nm_compute_sMs(m, st)) != NM_OK) break;
        if ((s = nm_pipe_setup(m)) != NM_OK) break;
        if (desc->terms & NM_TERM_DEMAG) {
            s = m->f64 ? setup_tables<double>(m, st) : setup_tables<float>(m, st);
            if (s != NM_OK) break;
            if ((s = nm_build_tensor(m, st)) != NM_OK) break;
            // the tensor setup used the Runge-Kutta region as scratch
            if (cudaMemsetAsync(m->K[0], 0, (char *)m->Q - (char *)m->K[0], st) != cudaSuccess) {
                nm_set_error("cudaMemsetAsync failed");
                s = NM_ECUDA;
                break;
            }
        }
        if (cudaStreamSynchronize(st) != cudaSuccess) {
            nm_set_error("nm_mesh_create: %s", cudaGetErrorString(cudaGetLastError()));
            s = NM_ECUDA;
        }
    } while (0);
    if (s != NM_OK) {
        delete m;
        return s;
    }
    // the pointers in desc are not kept
    m->desc.Ms = m->desc.A = m->desc.Ku = m->desc.D = m->desc.Kc = nullptr;
    *out = m;
    return NM_OK;
}

extern "C" nm_status nm_mesh_destroy(nm_mesh *mesh)
{
    if (mesh) {
        for (int i = 0; i < mesh->prof_ev_made; ++i) {
            cudaEventDestroy(mesh->prof_ev[i][0]);
            cudaEventDestroy(mesh->prof_ev[i][1]);
        }
        for (int i = 0; i < NM_GRAPH_SLOTS; ++i)
            if (mesh->step_graph[i].exec) cudaGraphExecDestroy(mesh->step_graph[i].exec);
        if (mesh->cap_stream) cudaStreamDestroy(mesh->cap_stream);
    }
    delete mesh;
    return NM_OK;
}

static const char *const kClassNames[NM_K_COUNT] = {"x_fwd", "y_fwd", "mid", "y_inv", "x_inv",
                                                    "node", "adj_cell", "lincomb", "other",
                                                    "node_rk", "node_adj"};

extern "C" int nm_profile_class_count(void) { return NM_K_COUNT; }

extern "C" const char *nm_profile_class_name(int cls)
{
    return cls >= 0 && cls < NM_K_COUNT ? kClassNames[cls] : "";
}

extern "C" nm_status nm_profile_begin(nm_mesh *mesh)
{
    if (!mesh) { nm_set_error("NULL argument"); return NM_EINVAL; }
    mesh->prof_on = true;
    mesh->prof_n = 0;
    mesh->prof_dropped = 0;
    return NM_OK;
}

extern "C" nm_status nm_profile_end(nm_mesh *mesh, void *stream, double *ms_host, long long *count_host)
{
    if (!mesh || !ms_host || !count_host) { nm_set_error("NULL argument"); return NM_EINVAL; }
    mesh->prof_on = false;
    NM_CUDA_TRY(cudaSetDevice(mesh->desc.device));
    NM_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    for (int c = 0; c < NM_K_COUNT; ++c) { ms_host[c] = 0.0; count_host[c] = 0; }
    for (int i = 0; i < mesh->prof_n; ++i) {
        float ms = 0.f;
        NM_CUDA_TRY(cudaEventElapsedTime(&ms, mesh->prof_ev[i][0], mesh->prof_ev[i][1]));
        ms_host[mesh->prof_cls[i]] += ms;
        count_host[mesh->prof_cls[i]]++;
    }
    mesh->prof_n = 0;
    return NM_OK;
}

extern "C" long long nm_launch_count(const nm_mesh *mesh) { return mesh ? mesh->launches : 0; }

extern "C" long long nm_profile_dropped(const nm_mesh *mesh) { return mesh ? mesh->prof_dropped : 0; }

extern "C" int nm_debug_demag_path(const nm_mesh *mesh)
{
    if (!mesh || !mesh->fast.on) return 0;
    return mesh->fast.embed ? 2 : 1;
}

extern "C" nm_status nm_debug_get_tensor(nm_mesh *mesh, double *N_host)
{
    if (!mesh || !N_host) { nm_set_error("NULL argument"); return NM_EINVAL; }
    if (!mesh->Nreal) { nm_set_error("mesh has no demag term"); return NM_EINVAL; }
    NM_CUDA_TRY(cudaSetDevice(mesh->desc.device));
    NM_CUDA_TRY(cudaMemcpy(N_host, mesh->Nreal, 6 * mesh->g.cells * sizeof(double), cudaMemcpyDeviceToHost));
    return NM_OK;
}

extern "C" nm_status nm_debug_get_cell_field(nm_mesh *mesh, void *Hc_out, void *stream)
{
    if (!mesh || !Hc_out) { nm_set_error("NULL argument"); return NM_EINVAL; }
    if (!mesh->Hc1 || !mesh->hc1_valid) { nm_set_error("no cell demag field has been computed"); return NM_EINVAL; }
    NM_CUDA_TRY(cudaSetDevice(mesh->desc.device));
    NM_CUDA_TRY(cudaMemcpyAsync(Hc_out, mesh->Hc1, 3 * mesh->g.cells * mesh->esz, cudaMemcpyDeviceToDevice,
                                (cudaStream_t)stream));
    return NM_OK;
}

// ---- field evaluation --------------------------------------------------------------------------
namespace {

// Constant part of the node-kernel arguments for this mesh at time t.
template <typename T>
void base_args(const nm_mesh *m, double t, const nm_zeeman *z, unsigned terms, NmLocalArgs<T> *a)
{
    memset(a, 0, sizeof(*a));
    a->g = m->g;
    a->Ms = (const T *)m->Ms;
    a->A = (const T *)m->A;
    a->Ku = (const T *)m->Ku;
    a->sMs = (const T *)m->sMs;
    a->terms = terms;
    const double *dx = m->desc.cell_size;
    const double V = dx[0] * dx[1] * dx[2];
    for (int e = 0; e < 8; ++e) {
        // vertices differ along axis d iff bit d of e is set: 1-D entries K1 = +-1, M1 = 1/3 or 1/6
        double wm = V, wk = 0.0;
        for (int d = 0; d < 3; ++d) wm *= ((e >> d) & 1) ? 1.0 / 6.0 : 1.0 / 3.0;
        for (int d = 0; d < 3; ++d) {
            double term = (((e >> d) & 1) ? -1.0 : 1.0) / (dx[d] * dx[d]);
            for (int f = 0; f < 3; ++f)
                if (f != d) term *= ((e >> f) & 1) ? 1.0 / 6.0 : 1.0 / 3.0;
            wk += term;
        }
        a->wK[e] = (T)(V * wk);
        a->wM[e] = (T)wm;
    }
    for (int j = 0; j < 3; ++j) a->kax[j] = (T)m->desc.ku_axis[j];
    a->mu0 = (T)NM_MU0;
    a->mu0V8 = (T)(NM_MU0 * V / 8.0);
    if ((terms & NM_TERM_ZEEMAN) && z) {
        a->h_static = (const T *)z->h_static;
        a->h_pulse = (const T *)z->h_pulse;
        a->amp = (T)(z->amp ? z->amp(t, z->user) : 1.0);
        for (int j = 0; j < 3; ++j) a->hu[j] = (T)z->h_uniform[j];
    }
    // separable kernel: uniform A and Ku (anisotropy off counts as uniform)
    const bool an_on = (terms & NM_TERM_ANISO) != 0;
    a->sep = (m->uni_A && (m->uni_Ku || !an_on)) ? 1 : 0;
    if (m->g.zs == 0) a->sep = 0;                                // reduced basis: the 27-point kernel with zero strides
    if (m->dbg_node_path == 1) a->sep = 0;                       // test switch, read once at nm_mesh_create
    else if (m->dbg_node_path == 2 && a->sep) a->sep = 2;
    a->cex = (terms & NM_TERM_EXCHANGE) ? (T)(16.0 * m->desc.A_scalar / NM_MU0) : (T)0;
    a->cku = an_on ? (T)(16.0 * m->desc.Ku_scalar / NM_MU0) : (T)0;
    for (int d = 0; d < 3; ++d) a->idx2[d] = (T)(1.0 / (dx[d] * dx[d]));
    a->ms_uni = m->uni_Ms ? (T)m->desc.Ms_scalar : (T)0;
    const double gp = m->desc.gamma / (1.0 + m->desc.alpha * m->desc.alpha);
    a->gp = (T)gp;
    a->agp = (T)(m->desc.alpha * gp);
}

// Demag convolution of `fld` into Hc (if the term is on) and the matching pointer for the node kernel.
template <typename T>
nm_status demag_part(nm_mesh *m, const T *fld, T *Hc, const T **Hc_arg, cudaStream_t st)
{
    *Hc_arg = nullptr;
    if (m->desc.terms & NM_TERM_DEMAG) {
        NM_TRY(nm_demag_conv<T>(m, fld, Hc, st));
        *Hc_arg = Hc;
    }
    return NM_OK;
}

// Field of the further local terms (NM_TERM_DMI, NM_TERM_CUBIC, NM_TERM_RKKY) of `fld` into the mesh's Xs array,
// which the node kernel then adds to H.  about != null (adjoint pass 2): the cubic term's derivative at `about`
// applied to fld; the other terms are linear and act on fld as they are.
template <typename T>
nm_status extra_part(nm_mesh *m, const T *fld, const T **hadd_arg, cudaStream_t st, const T *about = nullptr)
{
    if (!m->Xs) return NM_OK;
    NmExtraArgs<T> x;
    memset(&x, 0, sizeof(x));
    x.g = m->g;
    x.fld = fld;
    x.about = about;
    x.Ms = (const T *)m->Ms;
    x.D = (const T *)m->Dmi;
    x.Kc = (const T *)m->Kcub;
    x.out = (T *)m->Xs;
    const double *dx = m->desc.cell_size;
    const double V = dx[0] * dx[1] * dx[2];
    x.V = (T)V;
    x.mu0V8 = (T)(NM_MU0 * V / 8.0);
    for (int d = 0; d < 3; ++d) x.idx[d] = (T)(1.0 / dx[d]);
    x.dmi_kind = m->desc.dmi_kind;
    x.dmi_normal = m->desc.dmi_normal;
    for (int q = 0; q < 9; ++q) x.cax[q] = (T)m->desc.cubic_axes[q];
    x.rkky_JA = (m->desc.terms & NM_TERM_RKKY) ? (T)(m->desc.rkky_J * dx[0] * dx[1]) : (T)0;
    x.rkky_za = m->desc.rkky_planes[0];
    x.rkky_zb = m->desc.rkky_planes[1];
    NM_TRY(nm_launch_extra<T>(m, x, st));
    *hadd_arg = (const T *)m->Xs;
    return NM_OK;
}

template <typename T>
nm_status eval_simple(nm_mesh *m, double t, const T *fld, const nm_zeeman *z, T *out, int mode,
                      cudaStream_t st)
{
    NmLocalArgs<T> a;
    base_args<T>(m, t, z, m->desc.terms, &a);
    a.fld = fld;
    NM_TRY(extra_part<T>(m, fld, &a.hadd, st));
    NM_TRY(demag_part<T>(m, fld, (T *)m->Hc1, &a.Hc, st));
    m->hc1_valid = a.Hc != nullptr;
    a.mode = mode;
    a.out = out;
    return nm_launch_node<T>(m, a, st);
}

// One Runge-Kutta stage: k = f(t, fld) with the stage combination fused into the node kernel.
template <typename T>
nm_status eval_stage(nm_mesh *m, double t, const T *fld, const nm_zeeman *z, const NmRkArgs<T> &rk,
                     cudaStream_t st)
{
    NmLocalArgs<T> a;
    base_args<T>(m, t, z, m->desc.terms, &a);
    a.fld = fld;
    NM_TRY(extra_part<T>(m, fld, &a.hadd, st));
    NM_TRY(demag_part<T>(m, fld, (T *)m->Hc1, &a.Hc, st));
    m->hc1_valid = a.Hc != nullptr;
    a.mode = NM_MODE_RK;
    a.rk = rk;
    return nm_launch_node<T>(m, a, st);
}

template <typename T>
nm_status rk4_step(nm_mesh *m, double t, double dt, T *y, const nm_zeeman *z, int renorm, cudaStream_t st)
{
    // Classical RK4 without stored derivatives: the stage states carry them,
    //   Y0 = y + dt/2 k1,  Y1 = y + dt/2 k2,  Y2 = y + dt k3
    //   y + dt/6 (k1 + 2 k2 + 2 k3 + k4) = -1/3 y + 1/3 Y0 + 2/3 Y1 + 1/3 Y2 + dt/6 k4,
    // so a stage writes one nodal vector and the last one reads y, Y0, Y1 (Y2 is its own input).
    T *Y0 = (T *)m->Y[0], *Y1 = (T *)m->Y[1], *Y2 = (T *)m->K[0];
    NmRkArgs<T> r;
    memset(&r, 0, sizeof(r));
    r.y0 = y;
    r.dt = (T)dt;
    r.cself = (T)0.5; r.ynext = Y0;
    NM_TRY(eval_stage<T>(m, t, y, z, r, st));
    r.ynext = Y1;
    NM_TRY(eval_stage<T>(m, t + 0.5 * dt, Y0, z, r, st));
    r.cself = (T)1; r.ynext = Y2;
    NM_TRY(eval_stage<T>(m, t + 0.5 * dt, Y1, z, r, st));
    r.nstate = 2;
    r.sprev[0] = Y0; r.sprev[1] = Y1;
    r.bs[0] = (T)(-1.0 / 3.0); r.bs[1] = (T)(1.0 / 3.0); r.bs[2] = (T)(2.0 / 3.0); r.bs[3] = (T)(1.0 / 3.0);
    r.cself = (T)(1.0 / 6.0);
    r.ynext = y;
    r.renorm = renorm;
    return eval_stage<T>(m, t + dt, Y2, z, r, st);
}

// Dormand-Prince 5(4) (Dormand & Prince 1980; "Dormand-Prince method")
const double DP_C[7] = {0.0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0};
const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0.0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
const double DP_B5[7] = {35.0 / 384, 0.0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0.0};
const double DP_B4[7] = {5179.0 / 57600, 0.0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200,
                         187.0 / 2100, 1.0 / 40};

template <typename T>
nm_status dopri5_step(nm_mesh *m, double t, double dt, T *y, const nm_zeeman *z, int renorm,
                      double rtol, double atol, cudaStream_t st)
{
    T *Yb[2] = {(T *)m->Y[0], (T *)m->Y[1]};
    const T *fld = y;
    for (int s = 0; s < 7; ++s) {
        NmRkArgs<T> r;
        memset(&r, 0, sizeof(r));
        r.y0 = y;
        r.dt = (T)dt;
        r.kstore = s < 6 ? (T *)m->K[s] : nullptr;
        r.nprev = s;
        for (int j = 0; j < s; ++j) r.kprev[j] = (const T *)m->K[j];
        if (s < 6) {
            // next stage state (s < 5) or the fifth-order solution y5 (s = 5: row 6 of A equals b5)
            for (int j = 0; j < s; ++j) r.cprev[j] = (T)DP_A[s + 1][j];
            r.cself = (T)DP_A[s + 1][s];
            r.ynext = Yb[s & 1];
        } else {
            for (int j = 0; j < 6; ++j) r.eprev[j] = (T)(DP_B5[j] - DP_B4[j]);
            r.eself = (T)(DP_B5[6] - DP_B4[6]);
            r.want_err = 1;
            r.rtol = (T)rtol;
            r.atol = (T)atol;
            r.partials = m->partials;
        }
        NM_TRY(eval_stage<T>(m, t + DP_C[s] * dt, fld, z, r, st));
        if (s < 6) fld = Yb[s & 1];
    }
    NM_TRY(nm_launch_err_final(m, m->last_partials, 3.0 * (double)m->g.nodes, st));
    // y5 lives in Yb[5 & 1]
    return nm_launch_commit<T>(m, y, Yb[1], m->partials + m->n_partials, renorm, st);
}

// (f, -(df/dm)^T a, -(df/dMs)^T a): reading C7, two demag convolutions and two node passes.
template <typename T>
nm_status adjoint_eval(nm_mesh *m, double t, const T *mm, const T *av, const nm_zeeman *z, T *f_out,
                       T *dadt, T *dudt, cudaStream_t st)
{
    NmLocalArgs<T> a;
    base_args<T>(m, t, z, m->desc.terms, &a);
    a.fld = mm;
    NM_TRY(extra_part<T>(m, mm, &a.hadd, st));
    NM_TRY(demag_part<T>(m, mm, (T *)m->Hc1, &a.Hc, st));
    m->hc1_valid = a.Hc != nullptr;
    a.mode = NM_MODE_ADJ1;
    a.out = f_out;
    a.adj = av;
    a.Q = (T *)m->Q;
    a.W = (T *)m->W;
    a.dadt = dadt;
    NM_TRY(nm_launch_node<T>(m, a, st));
    // Hlin^T b = (S Ms) o Hlin(q): same operators on q = b / (S Ms), no Zeeman term
    NmLocalArgs<T> b;
    base_args<T>(m, t, nullptr, m->desc.terms & ~(unsigned)NM_TERM_ZEEMAN, &b);
    b.fld = (const T *)m->Q;
    NM_TRY(extra_part<T>(m, (const T *)m->Q, &b.hadd, st, mm));   // cubic: -Hess E(m) q / L, the rest linear in q
    NM_TRY(demag_part<T>(m, (const T *)m->Q, (T *)m->Hc2, &b.Hc, st));
    b.mode = NM_MODE_ADJ2;
    b.dadt = dadt;
    NM_TRY(nm_launch_node<T>(m, b, st));
    if (dudt) {
        NmAdjCellArgs<T> c;
        memset(&c, 0, sizeof(c));
        c.g = m->g;
        c.m = mm;
        c.Q = (const T *)m->Q;
        c.W = (const T *)m->W;
        c.Hc1 = a.Hc;
        c.Hc2 = b.Hc;
        c.h_static = a.h_static;
        c.h_pulse = a.h_pulse;
        c.amp = a.amp;
        for (int j = 0; j < 3; ++j) c.hu[j] = a.hu[j];
        for (int e = 0; e < 8; ++e) {
            double wm = 8.0;   // (8/V) * V prod_d M1
            for (int d = 0; d < 3; ++d) wm *= ((e >> d) & 1) ? 1.0 / 6.0 : 1.0 / 3.0;
            c.wM8V[e] = (T)wm;
        }
        c.terms = (m->desc.terms & NM_TERM_ZEEMAN) && z ? m->desc.terms : (m->desc.terms & ~(unsigned)NM_TERM_ZEEMAN);
        c.dudt = dudt;
        c.red = (T)nm_red_scale(m);
        NM_TRY(nm_launch_adj_cell<T>(m, c, st));
    }
    return NM_OK;
}

// VJPs with respect to the cell-wise A and Ku for the state (mm, av): write (accumulate == 0) or
// u_X += coef g_X.
template <typename T>
nm_status mat_grad(nm_mesh *m, const T *mm, const T *av, T *uA, T *uKu, double coef, int accumulate,
                   cudaStream_t st)
{
    if (!uA && !uKu) return NM_OK;
    NmLocalArgs<T> la;
    base_args<T>(m, 0.0, nullptr, m->desc.terms, &la);
    NmMatGradArgs<T> g;
    memset(&g, 0, sizeof(g));
    g.g = m->g;
    g.m = mm;
    g.a = av;
    g.sMs = (const T *)m->sMs;
    g.u_A = uA;
    g.u_Ku = uKu;
    for (int e = 0; e < 8; ++e) { g.wK[e] = la.wK[e]; g.wM[e] = la.wM[e]; }
    for (int j = 0; j < 3; ++j) g.kax[j] = la.kax[j];
    g.gp = la.gp;
    g.agp = la.agp;
    const double V = m->desc.cell_size[0] * m->desc.cell_size[1] * m->desc.cell_size[2];
    g.invL = (T)(8.0 * nm_red_scale(m) / (NM_MU0 * V));     // 2^D / (mu0 V)
    g.coef = (T)coef;
    g.accumulate = accumulate;
    g.ex_on = (m->desc.terms & NM_TERM_EXCHANGE) != 0;
    g.an_on = (m->desc.terms & NM_TERM_ANISO) != 0;
    return nm_launch_mat_grad<T>(m, g, st);
}

template <typename T>
nm_status adjoint_rk4(nm_mesh *m, double t, double dt, T *mm, T *av, T *u, double *uh, T *uA, T *uKu, T *uhn,
                      const nm_zeeman *z, int renorm, cudaStream_t st)
{
    const double gp_h = m->desc.gamma / (1.0 + m->desc.alpha * m->desc.alpha);
    const bool want_h = uh && (m->desc.terms & NM_TERM_ZEEMAN);
    const long long nv = 3 * m->g.nodes, nc = m->g.cells, nn = m->g.nodes;
    T *F = (T *)m->K[0], *DA = (T *)m->K[1], *AM = (T *)m->K[2], *AA = (T *)m->K[3];
    T *Ym = (T *)m->Y[0], *Ya = (T *)m->Y[1];
    T *DU = (T *)m->Uc[0], *AU = (T *)m->Uc[1];
    const double h = -dt;
    const double w[4] = {h / 6, h / 3, h / 3, h / 6};
    const double cn[3] = {0.5 * h, 0.5 * h, h};     // next stage state = y + cn * k
    const double ts[4] = {t, t + 0.5 * h, t + 0.5 * h, t + h};
    const T *sm = mm, *sa = av;
    for (int s = 0; s < 4; ++s) {
        NM_TRY(adjoint_eval<T>(m, ts[s], sm, sa, z, F, DA, DU, st));
        // u_h += w_s (-(df/dh)^T a) of this stage (reads the stage state before it is overwritten)
        if (want_h) NM_TRY(nm_launch_hext_grad<T>(m, sm, sa, gp_h, m->desc.alpha * gp_h, w[s], uh, st));
        if (uhn && (m->desc.terms & NM_TERM_ZEEMAN)) {      // u_hn += w_s Z(b / L): q = b / (S Ms) is in Q after the adjoint pass
            NmLocalArgs<T> la;
            base_args<T>(m, 0.0, nullptr, m->desc.terms, &la);
            NM_TRY(nm_launch_hnodal_grad<T>(m, la, (const T *)m->Q, sm, sa, w[s], 1, uhn, st));
        }
        NM_TRY(mat_grad<T>(m, sm, sa, uA, uKu, w[s], 1, st));
        const T ws = (T)w[s];
        if (s < 3) {
            // accumulators (the first stage starts them from the state) and the next stage state
            const T c = (T)cn[s];
            const NmLinOp<T> ops[5] = {{AM, s == 0 ? mm : AM, F, ws, nv, 0},
                                       {AA, s == 0 ? av : AA, DA, ws, nv, 0},
                                       {AU, s == 0 ? u : AU, DU, ws, nc, 0},
                                       {Ym, mm, F, c, nv, 0},
                                       {Ya, av, DA, c, nv, 0}};
            NM_TRY(nm_lincomb_batch<T>(m, ops, 5, st));
            sm = Ym;
            sa = Ya;
        } else {
            const NmLinOp<T> ops[3] = {{mm, AM, F, ws, nv, renorm ? nn : 0},
                                       {av, AA, DA, ws, nv, 0},
                                       {u, AU, DU, ws, nc, 0}};
            NM_TRY(nm_lincomb_batch<T>(m, ops, 3, st));
        }
    }
    return NM_OK;
}

// Whole-step graph replay.  A step whose launch sequence is fixed by `key` (no host callback, no
// per-launch timing) runs eagerly the first time; when the same key arrives again the sequence is
// captured once on the mesh's capture stream (capture executes nothing) and from then on replayed
// with one cudaGraphLaunch on the caller's stream.  `issue(stream)` enqueues the step.
template <typename F>
nm_status run_step(nm_mesh *m, int slot, const nm_zeeman *z, NmStepKey key, cudaStream_t st, F issue)
{
    if (!m->graph_on || m->prof_on || (z && z->amp)) return issue(st);
    {
        // the caller is capturing this stream into a graph of their own: plain launches go into it
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); return issue(st); }
        if (cs != cudaStreamCaptureStatusNone) return issue(st);
    }
    key.kind = slot;
    key.epoch = m->graph_epoch;
    key.has_z = z != nullptr;
    if (z) {
        key.hs = z->h_static;
        key.hp = z->h_pulse;
        for (int j = 0; j < 3; ++j) key.hu[j] = z->h_uniform[j];
    }
    NmStepGraph &sg = m->step_graph[slot];
    if (sg.seen && memcmp(&sg.key, &key, sizeof(key)) == 0) {
        if (!sg.exec) {
            if (!m->cap_stream) NM_CUDA_TRY(cudaStreamCreateWithFlags(&m->cap_stream, cudaStreamNonBlocking));
            NM_CUDA_TRY(cudaStreamBeginCapture(m->cap_stream, cudaStreamCaptureModeRelaxed));
            const long long before = m->launches;
            const nm_status s = issue(m->cap_stream);
            cudaGraph_t graph = nullptr;
            const cudaError_t e = cudaStreamEndCapture(m->cap_stream, &graph);
            sg.launches = m->launches - before;
            m->launches = before;
            if (s != NM_OK || e != cudaSuccess || !graph) {
                if (graph) cudaGraphDestroy(graph);
                cudaGetLastError();
                if (s != NM_OK) return s;
                m->graph_on = false;            // capture not possible here: stay on plain launches
                return issue(st);
            }
            const cudaError_t ei = cudaGraphInstantiate(&sg.exec, graph, 0);
            cudaGraphDestroy(graph);
            if (ei != cudaSuccess) {
                sg.exec = nullptr;
                cudaGetLastError();
                m->graph_on = false;
                return issue(st);
            }
        }
        NM_CUDA_TRY(cudaGraphLaunch(sg.exec, st));
        m->launches += sg.launches;
        return NM_OK;
    }
    if (sg.exec) {
        cudaGraphExecDestroy(sg.exec);
        sg.exec = nullptr;
    }
    sg.key = key;
    sg.seen = true;
    return issue(st);
}

nm_status check_call(nm_mesh *mesh, const void *p0, const void *p1)
{
    if (!mesh || !p0 || !p1) { nm_set_error("NULL argument"); return NM_EINVAL; }
    NM_CUDA_TRY(cudaSetDevice(mesh->desc.device));
    return NM_OK;
}

} // namespace

extern "C" nm_status nm_heff(nm_mesh *mesh, double t, const void *m, const nm_zeeman *zeeman, void *H_out,
                             void *stream)
{
    NM_TRY(check_call(mesh, m, H_out));
    cudaStream_t st = (cudaStream_t)stream;
    return mesh->f64 ? eval_simple<double>(mesh, t, (const double *)m, zeeman, (double *)H_out, NM_MODE_H, st)
                     : eval_simple<float>(mesh, t, (const float *)m, zeeman, (float *)H_out, NM_MODE_H, st);
}

extern "C" nm_status nm_llg_rhs(nm_mesh *mesh, double t, const void *m, const nm_zeeman *zeeman,
                                void *dmdt_out, void *stream)
{
    NM_TRY(check_call(mesh, m, dmdt_out));
    cudaStream_t st = (cudaStream_t)stream;
    return mesh->f64 ? eval_simple<double>(mesh, t, (const double *)m, zeeman, (double *)dmdt_out, NM_MODE_RHS, st)
                     : eval_simple<float>(mesh, t, (const float *)m, zeeman, (float *)dmdt_out, NM_MODE_RHS, st);
}

extern "C" nm_status nm_rk_step(nm_mesh *mesh, nm_scheme scheme, double t, double dt, void *m_inout,
                                const nm_zeeman *zeeman, int renormalise, double rtol, double atol,
                                double *err_norm_host, void *stream)
{
    NM_TRY(check_call(mesh, m_inout, m_inout));
    cudaStream_t st = (cudaStream_t)stream;
    NmStepKey key;
    memset(&key, 0, sizeof(key));
    key.dt = dt;
    key.renorm = renormalise;
    key.p[0] = m_inout;
    if (scheme == NM_RK4) {
        if (err_norm_host) *err_norm_host = 0.0;
        return run_step(mesh, NM_GRAPH_RK4, zeeman, key, st, [&](cudaStream_t s) {
            return mesh->f64 ? rk4_step<double>(mesh, t, dt, (double *)m_inout, zeeman, renormalise, s)
                             : rk4_step<float>(mesh, t, dt, (float *)m_inout, zeeman, renormalise, s);
        });
    }
    if (scheme == NM_DOPRI5) {
        if (!(rtol >= 0) || !(atol >= 0) || (rtol == 0 && atol == 0)) {
            nm_set_error("rtol / atol must be non-negative and not both zero");
            return NM_EINVAL;
        }
        key.rtol = rtol;
        key.atol = atol;
        // the launches replay; the read-back of the error norm stays outside the graph
        NM_TRY(run_step(mesh, NM_GRAPH_DOPRI5, zeeman, key, st, [&](cudaStream_t s) {
            return mesh->f64 ? dopri5_step<double>(mesh, t, dt, (double *)m_inout, zeeman, renormalise, rtol,
                                                   atol, s)
                             : dopri5_step<float>(mesh, t, dt, (float *)m_inout, zeeman, renormalise, rtol,
                                                  atol, s);
        }));
        if (err_norm_host) {
            NM_CUDA_TRY(cudaMemcpyAsync(err_norm_host, mesh->partials + mesh->n_partials, sizeof(double),
                                        cudaMemcpyDeviceToHost, st));
            NM_CUDA_TRY(cudaStreamSynchronize(st));
        }
        return NM_OK;
    }
    nm_set_error("unknown scheme %d", (int)scheme);
    return NM_EINVAL;
}

extern "C" nm_status nm_llg_adjoint_rhs(nm_mesh *mesh, double t, const void *m, const void *a,
                                        const nm_zeeman *zeeman, void *dmdt_out, void *dadt_out,
                                        void *dudt_Ms_out, void *stream)
{
    NM_TRY(check_call(mesh, m, a));
    if (!dadt_out) { nm_set_error("dadt_out is NULL"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    return mesh->f64 ? adjoint_eval<double>(mesh, t, (const double *)m, (const double *)a, zeeman,
                                            (double *)dmdt_out, (double *)dadt_out, (double *)dudt_Ms_out, st)
                     : adjoint_eval<float>(mesh, t, (const float *)m, (const float *)a, zeeman,
                                           (float *)dmdt_out, (float *)dadt_out, (float *)dudt_Ms_out, st);
}

namespace {
nm_status adjoint_rk4_entry(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout, void *u_inout,
                            double *u_h_inout, void *u_A, void *u_Ku, void *u_hn, const nm_zeeman *zeeman,
                            int renormalise, void *stream)
{
    NM_TRY(check_call(mesh, m_inout, a_inout));
    if (!u_inout) { nm_set_error("u_inout is NULL"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    NmStepKey key;
    memset(&key, 0, sizeof(key));
    key.dt = dt;
    key.renorm = renormalise;
    key.p[0] = m_inout;
    key.p[1] = a_inout;
    key.p[2] = u_inout;
    key.p[3] = u_h_inout;
    key.p[4] = u_A;
    key.p[5] = u_Ku;
    key.p[6] = u_hn;
    return run_step(mesh, NM_GRAPH_ADJ_RK4, zeeman, key, st, [&](cudaStream_t s) {
        return mesh->f64 ? adjoint_rk4<double>(mesh, t, dt, (double *)m_inout, (double *)a_inout,
                                               (double *)u_inout, u_h_inout, (double *)u_A, (double *)u_Ku,
                                               (double *)u_hn, zeeman, renormalise, s)
                         : adjoint_rk4<float>(mesh, t, dt, (float *)m_inout, (float *)a_inout,
                                              (float *)u_inout, u_h_inout, (float *)u_A, (float *)u_Ku,
                                              (float *)u_hn, zeeman, renormalise, s);
    });
}
} // namespace

extern "C" nm_status nm_adjoint_rk4_step(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                                         void *u_inout, const nm_zeeman *zeeman, int renormalise, void *stream)
{
    return adjoint_rk4_entry(mesh, t, dt, m_inout, a_inout, u_inout, nullptr, nullptr, nullptr, nullptr, zeeman,
                             renormalise, stream);
}

extern "C" nm_status nm_adjoint_rk4_step_hext(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                                              void *u_inout, double *u_h_inout, const nm_zeeman *zeeman,
                                              int renormalise, void *stream)
{
    if (!u_h_inout) { nm_set_error("u_h_inout is NULL"); return NM_EINVAL; }
    return adjoint_rk4_entry(mesh, t, dt, m_inout, a_inout, u_inout, u_h_inout, nullptr, nullptr, nullptr, zeeman,
                             renormalise, stream);
}

extern "C" nm_status nm_adjoint_rk4_step_ex(nm_mesh *mesh, double t, double dt, void *m_inout, void *a_inout,
                                            void *u_inout, const nm_adjoint_extra *extra,
                                            const nm_zeeman *zeeman, int renormalise, void *stream)
{
    if (!extra) { nm_set_error("extra is NULL"); return NM_EINVAL; }
    return adjoint_rk4_entry(mesh, t, dt, m_inout, a_inout, u_inout, extra->u_h, extra->u_A, extra->u_Ku,
                             extra->u_hn, zeeman, renormalise, stream);
}

extern "C" nm_status nm_llg_adjoint_rhs_hnodal(nm_mesh *mesh, const void *m, const void *a, void *dudt_hn_out,
                                               void *stream)
{
    NM_TRY(check_call(mesh, m, a));
    if (!dudt_hn_out) { nm_set_error("dudt_hn_out is NULL"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    if (!(mesh->desc.terms & NM_TERM_ZEEMAN)) {
        NM_CUDA_TRY(cudaMemsetAsync(dudt_hn_out, 0, 3 * mesh->g.nodes * mesh->esz, st));
        return NM_OK;
    }
    if (mesh->f64) {
        NmLocalArgs<double> la;
        base_args<double>(mesh, 0.0, nullptr, mesh->desc.terms, &la);
        return nm_launch_hnodal_grad<double>(mesh, la, nullptr, (const double *)m, (const double *)a, 1.0, 0,
                                             (double *)dudt_hn_out, st);
    }
    NmLocalArgs<float> la;
    base_args<float>(mesh, 0.0, nullptr, mesh->desc.terms, &la);
    return nm_launch_hnodal_grad<float>(mesh, la, nullptr, (const float *)m, (const float *)a, 1.0, 0,
                                        (float *)dudt_hn_out, st);
}

extern "C" nm_status nm_llg_adjoint_rhs_materials(nm_mesh *mesh, const void *m, const void *a, void *dudt_A_out,
                                                  void *dudt_Ku_out, void *stream)
{
    NM_TRY(check_call(mesh, m, a));
    if (!dudt_A_out && !dudt_Ku_out) { nm_set_error("both outputs are NULL"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    return mesh->f64 ? mat_grad<double>(mesh, (const double *)m, (const double *)a, (double *)dudt_A_out,
                                        (double *)dudt_Ku_out, 1.0, 0, st)
                     : mat_grad<float>(mesh, (const float *)m, (const float *)a, (float *)dudt_A_out,
                                       (float *)dudt_Ku_out, 1.0, 0, st);
}

extern "C" nm_status nm_llg_adjoint_rhs_hext(nm_mesh *mesh, const void *m, const void *a, double *dudt_h_out,
                                             void *stream)
{
    NM_TRY(check_call(mesh, m, a));
    if (!dudt_h_out) { nm_set_error("dudt_h_out is NULL"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    NM_CUDA_TRY(cudaMemsetAsync(dudt_h_out, 0, 3 * sizeof(double), st));
    if (!(mesh->desc.terms & NM_TERM_ZEEMAN)) return NM_OK;
    const double gp = mesh->desc.gamma / (1.0 + mesh->desc.alpha * mesh->desc.alpha);
    return mesh->f64 ? nm_launch_hext_grad<double>(mesh, (const double *)m, (const double *)a, gp,
                                                   mesh->desc.alpha * gp, 1.0, dudt_h_out, st)
                     : nm_launch_hext_grad<float>(mesh, (const float *)m, (const float *)a, gp,
                                                  mesh->desc.alpha * gp, 1.0, dudt_h_out, st);
}

extern "C" nm_status nm_adjoint_add_objective(nm_mesh *mesh, void *a_inout, const void *dLdm, double scale,
                                              void *stream)
{
    NM_TRY(check_call(mesh, a_inout, dLdm));
    if (a_inout == dLdm) { nm_set_error("a_inout and dLdm overlap"); return NM_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const long long nv = 3 * mesh->g.nodes;
    if (mesh->f64) {
        const double c = scale;
        const double *src[1] = {(const double *)dLdm};
        return nm_lincomb<double>(mesh, (double *)a_inout, (const double *)a_inout, 1, src, &c, nv, 0, st);
    }
    const float c = (float)scale;
    const float *src[1] = {(const float *)dLdm};
    return nm_lincomb<float>(mesh, (float *)a_inout, (const float *)a_inout, 1, src, &c, nv, 0, st);
}
