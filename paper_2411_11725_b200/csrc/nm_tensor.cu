// Demagnetisation tensor setup (nm_mesh_create; not on the hot path).
//
// Reading C4: N(c - c') is the interaction tensor of two identical uniformly
// magnetised cuboids.  By definition
//     N_ij(R) = 1/(4 pi V) int_cell int_cell' (delta_ij/rho^3 - 3 rho_i rho_j/rho^5) d3r d3r',
//     rho = R + r - r',
// which for |R| >= 8 max(dx) is a smooth integrand.  The double volume integral reduces to one
// 3-D integral over u = r - r' with the triangle weight prod_d (dx_d - |u_d|); it is evaluated
// here in fp64 with Gauss-Legendre points on each half-interval (6 points: error < 1e-18
// absolute at 8 cell sizes; 4 and 3 points further out; tests/test_gpu_parity.py:
// test_tensor_matches_oracle holds every entry of five grids to 1e-13 of the oracle's binary128
// closed form, the 48^3 grid reaching all three orders).  No cancellation occurs, unlike the
// closed form whose fp64 evaluation loses every digit beyond ~100 cells.  Offsets closer than
// that come from the closed form in binary128 on the host (nm_newell_host.cpp).
//
// The spectrum N^(k) of the even/odd-extended tensor on the padded grid is real; it is obtained
// by direct cosine / sine sums per axis in fp64 (independent of the FFT kernels it will be used
// with), folded to one octant, scaled by 1/(P1 P2 P3) and rounded to the mesh dtype.
#include <cmath>
#include <vector>

#include "nm_internal.h"

namespace {

// Gauss-Legendre nodes / weights on [0,1]
__constant__ double c_gl_x[3][6] = {
    {0.11270166537925831148, 0.5, 0.88729833462074168852, 0, 0, 0},
    {0.06943184420297371239, 0.33000947820757186760, 0.66999052179242813240,
     0.93056815579702628761, 0, 0},
    {0.03376524289842398609, 0.16939530676686774317, 0.38069040695840154568,
     0.61930959304159845432, 0.83060469323313225683, 0.96623475710157601391}};
__constant__ double c_gl_w[3][6] = {
    {0.27777777777777777778, 0.44444444444444444444, 0.27777777777777777778, 0, 0, 0},
    {0.17392742256872692869, 0.32607257743127307131, 0.32607257743127307131,
     0.17392742256872692869, 0, 0},
    {0.08566224618958517252, 0.18038078652406930378, 0.23395696728634552369,
     0.23395696728634552369, 0.18038078652406930378, 0.08566224618958517252}};

__global__ void k_tensor_far(double *__restrict__ Nreal, int N1, int N2, int N3, double d1,
                             double d2, double d3, int b1, int b2, int b3, double r_mid,
                             double r_far)
{
    const long long cells = (long long)N1 * N2 * N3;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= cells) return;
    const int p1 = (int)(idx % N1);
    const int p2 = (int)((idx / N1) % N2);
    const int p3 = (int)(idx / ((long long)N1 * N2));
    if (p1 < b1 && p2 < b2 && p3 < b3) return;   // near box: closed form from the host
    const double X = p1 * d1, Y = p2 * d2, Z = p3 * d3;
    const double R = sqrt(X * X + Y * Y + Z * Z);
    const int rule = R < r_mid ? 2 : (R < r_far ? 1 : 0);
    const int n = rule == 2 ? 6 : (rule == 1 ? 4 : 3);
    double sxx = 0, syy = 0, szz = 0, sxy = 0, sxz = 0, syz = 0;
    for (int i = 0; i < 2 * n; ++i) {
        const double si = c_gl_x[rule][i % n];
        const double wi = c_gl_w[rule][i % n] * (1.0 - si);
        const double x = X + (i < n ? si : -si) * d1;
        for (int j = 0; j < 2 * n; ++j) {
            const double sj = c_gl_x[rule][j % n];
            const double wij = wi * c_gl_w[rule][j % n] * (1.0 - sj);
            const double y = Y + (j < n ? sj : -sj) * d2;
            for (int k = 0; k < 2 * n; ++k) {
                const double sk = c_gl_x[rule][k % n];
                const double w = wij * c_gl_w[rule][k % n] * (1.0 - sk);
                const double z = Z + (k < n ? sk : -sk) * d3;
                const double r2 = x * x + y * y + z * z;
                const double ir = rsqrt(r2);
                const double ir3 = ir * ir * ir;
                const double w3 = w * ir3;
                const double w5 = 3.0 * w3 * ir * ir;
                sxx += w3 - w5 * x * x;
                syy += w3 - w5 * y * y;
                szz += w3 - w5 * z * z;
                sxy -= w5 * x * y;
                sxz -= w5 * x * z;
                syz -= w5 * y * z;
            }
        }
    }
    // (1/V) prod_d dx_d^2 = V
    const double pref = d1 * d2 * d3 / (4.0 * 3.14159265358979323846264338327950288);
    Nreal[0 * cells + idx] = pref * sxx;
    Nreal[1 * cells + idx] = pref * syy;
    Nreal[2 * cells + idx] = pref * szz;
    Nreal[3 * cells + idx] = pref * sxy;
    Nreal[4 * cells + idx] = pref * sxz;
    Nreal[5 * cells + idx] = pref * syz;
}

__global__ void k_tensor_put_box(double *__restrict__ Nreal, const double *__restrict__ box,
                                 int N1, int N2, int N3, int b1, int b2, int b3)
{
    const long long nb = (long long)b1 * b2 * b3;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 6 * nb) return;
    const int a = (int)(idx / nb);
    const long long r = idx % nb;
    const int p1 = (int)(r % b1), p2 = (int)((r / b1) % b2), p3 = (int)(r / ((long long)b1 * b2));
    Nreal[((long long)a * N3 + p3) * N2 * N1 + (long long)p2 * N1 + p1] = box[idx];
}

// in: [6][outer][N][inner] -> out: [6][outer][K][inner]; even axis: n(0) + 2 sum n(x) cos(2 pi k x/P),
// odd axis: 2 sum n(x) sin(2 pi k x/P)  (the factor -i per odd axis is applied at the end).
__global__ void k_axis_sum(const double *__restrict__ in, double *__restrict__ out,
                           long long outer, int N, int K, long long inner, int P, int axis)
{
    const long long per = outer * K * inner;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 6 * per) return;
    const int a = (int)(idx / per);
    long long r = idx % per;
    const long long in_i = r % inner;
    r /= inner;
    const int k = (int)(r % K);
    const long long o = r / K;
    // component a = (xx,yy,zz,xy,xz,yz): odd along `axis` iff the axis is one of its two indices
    const bool odd = (a == 3 && (axis == 0 || axis == 1)) || (a == 4 && (axis == 0 || axis == 2)) ||
                     (a == 5 && (axis == 1 || axis == 2));
    const double *src = in + ((long long)a * outer + o) * N * inner + in_i;
    double acc = 0.0;
    int ph = 0;   // (k * x) mod P
    for (int x = 1; x < N; ++x) {
        ph += k;
        if (ph >= P) ph -= P;
        const double ang = 2.0 * (double)ph / (double)P;
        acc += src[(long long)x * inner] * (odd ? sinpi(ang) : cospi(ang));
    }
    double v = 2.0 * acc;
    if (!odd) v += src[0];
    if (odd && P == 1) v = 0.0;
    out[(((long long)a * outer + o) * K + k) * inner + in_i] = v;
}

template <typename T>
__global__ void k_tensor_store(const double *__restrict__ in, T *__restrict__ Nhat, int K1,
                               int K2, int K3, int C1p, double scale)
{
    const long long per = (long long)K3 * K2 * C1p;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 6 * per) return;
    const int a = (int)(idx / per);
    const long long r = idx % per;
    const int k1 = (int)(r % C1p);
    const long long row = r / C1p;
    double v = 0.0;
    if (k1 < K1) {
        v = in[((long long)a * K3 * K2 + row) * K1 + k1] * scale;
        if (a >= 3) v = -v;   // (-i)^2 from the two odd axes
    }
    Nhat[idx] = (T)v;
}

inline unsigned blocks_for(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

} // namespace

nm_status nm_build_tensor(nm_mesh *mesh, cudaStream_t st)
{
    const NmGeom &g = mesh->g;
    const double *dx = mesh->desc.cell_size;
    const double dmax = std::fmax(dx[0], std::fmax(dx[1], dx[2]));
    const double r_cut = 8.0 * dmax;
    int box[3];
    const int N[3] = {g.N1, g.N2, g.N3};
    for (int d = 0; d < 3; ++d) {
        int b = (int)std::ceil(r_cut / dx[d]) + 1;
        box[d] = b < N[d] ? b : N[d];
    }
    const size_t nb = (size_t)box[0] * box[1] * box[2];
    std::vector<double> near(6 * nb);
    if (nm_newell_near_box(box, dx, near.data(), 0) != 0) {
        nm_set_error("nm_newell_near_box failed");
        return NM_ENOMEM;
    }
    // scratch inside the (not yet used) Runge-Kutta region of the workspace
    const long long K1 = g.C1, K2 = g.K2, K3 = g.K3;
    double *s0 = (double *)mesh->K[0];
    double *s1 = s0 + 6 * K1 * K2 * K3;
    NM_CUDA_TRY(cudaMemcpyAsync(s0, near.data(), near.size() * sizeof(double),
                                cudaMemcpyHostToDevice, st));
    k_tensor_far<<<blocks_for(g.cells, 128), 128, 0, st>>>(mesh->Nreal, g.N1, g.N2, g.N3, dx[0],
                                                          dx[1], dx[2], box[0], box[1], box[2],
                                                          16.0 * dmax, 40.0 * dmax);
    k_tensor_put_box<<<blocks_for(6 * (long long)nb, 256), 256, 0, st>>>(
        mesh->Nreal, s0, g.N1, g.N2, g.N3, box[0], box[1], box[2]);
    NM_CUDA_TRY(cudaGetLastError());
    NM_CUDA_TRY(cudaStreamSynchronize(st));   // `near` must outlive the copy; s0 is reused below
    // x: [6][N3*N2][N1][1] -> [6][N3*N2][K1][1]
    k_axis_sum<<<blocks_for(6LL * g.N3 * g.N2 * K1, 256), 256, 0, st>>>(
        mesh->Nreal, s0, (long long)g.N3 * g.N2, g.N1, (int)K1, 1, g.P1, 0);
    // y: [6][N3][N2][K1] -> [6][N3][K2][K1]
    k_axis_sum<<<blocks_for(6LL * g.N3 * K2 * K1, 256), 256, 0, st>>>(s0, s1, g.N3, g.N2, (int)K2,
                                                                     K1, g.P2, 1);
    // z: [6][1][N3][K2*K1] -> [6][1][K3][K2*K1]
    k_axis_sum<<<blocks_for(6LL * K3 * K2 * K1, 256), 256, 0, st>>>(s1, s0, 1, g.N3, (int)K3,
                                                                   K2 * K1, g.P3, 2);
    const double scale = 1.0 / ((double)g.P1 * g.P2 * g.P3);
    const long long tot = 6LL * K3 * K2 * g.C1p;
    if (mesh->fast.on) {
        NM_TRY(nm_fast_store_tensor(mesh, s0, scale, st));
    } else if (mesh->f64)
        k_tensor_store<double><<<blocks_for(tot, 256), 256, 0, st>>>(s0, (double *)mesh->Nhat,
                                                                    (int)K1, (int)K2, (int)K3,
                                                                    g.C1p, scale);
    else
        k_tensor_store<float><<<blocks_for(tot, 256), 256, 0, st>>>(s0, (float *)mesh->Nhat,
                                                                   (int)K1, (int)K2, (int)K3,
                                                                   g.C1p, scale);
    NM_CUDA_TRY(cudaGetLastError());
    NM_CUDA_TRY(cudaStreamSynchronize(st));
    return NM_OK;
}
