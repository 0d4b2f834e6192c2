// Near-field part of the demagnetisation tensor, host side, __float128.
//
// Reading C4: interaction tensor of two identical uniformly magnetised cuboids
// ("homogeneously magnetized cuboidal simulation cells arranged on a regular grid",
// PAPER.md:181) in the Newell closed form.  The closed form is a triple second difference of
// an antiderivative that grows like R^3 while the result decays like R^-3, so it is only used
// for the box of offsets near the origin (where the dipole-kernel quadrature of nm_tensor.cu
// converges slowly) and evaluated in binary128 so that no digit is lost.
//
// Organisation differs from a lattice-then-difference scheme on purpose: the three 1-D second
// differences are expanded into the 27 signed corner evaluations per offset, with each distinct
// antiderivative value computed once per thread-owned slab and reused through a small cache.
#include <quadmath.h>

#include <algorithm>
#include <atomic>
#include <cstddef>
#include <thread>
#include <vector>

namespace {

typedef __float128 quad;

inline quad sq(quad v) { return v * v; }

// Second antiderivative pieces.  F2 is the diagonal generator, G2 the off-diagonal one.
quad F2(quad x, quad y, quad z)
{
    const quad xx = sq(x), yy = sq(y), zz = sq(z);
    const quad rr = xx + yy + zz;
    if (rr == 0) return 0;
    const quad r = sqrtq(rr);
    quad acc = (2 * xx - yy - zz) * r / 6;
    const quad pxz = xx + zz, pxy = xx + yy;
    if (pxz > 0 && y != 0) acc += (y / 2) * (zz - xx) * asinhq(y / sqrtq(pxz));
    if (pxy > 0 && z != 0) acc += (z / 2) * (yy - xx) * asinhq(z / sqrtq(pxy));
    if (x != 0 && y != 0 && z != 0) acc -= x * y * z * atanq((y * z) / (x * r));
    return acc;
}

quad G2(quad x, quad y, quad z)
{
    const quad xx = sq(x), yy = sq(y), zz = sq(z);
    const quad rr = xx + yy + zz;
    if (rr == 0) return 0;
    const quad r = sqrtq(rr);
    // every term carries a factor x or y, or an atan/asinh of 0: G2 is odd in x and in y
    if (x == 0 || y == 0) return 0;
    quad acc = -x * y * r / 3;
    const quad pxy = xx + yy, pyz = yy + zz, pxz = xx + zz;
    if (pxy > 0 && z != 0) acc += x * y * z * asinhq(z / sqrtq(pxy));
    if (pyz > 0 && x != 0) acc += (y / 6) * (3 * zz - yy) * asinhq(x / sqrtq(pyz));
    if (pxz > 0 && y != 0) acc += (x / 6) * (3 * zz - xx) * asinhq(y / sqrtq(pxz));
    if (z != 0) {
        acc -= (z * zz / 6) * atanq((x * y) / (z * r));
        if (y != 0) acc -= (z * yy / 2) * atanq((x * z) / (y * r));
        if (x != 0) acc -= (z * xx / 2) * atanq((y * z) / (x * r));
    }
    return acc;
}

struct Gen {
    int comp;
    quad d[3];
    quad operator()(long a, long b, long c) const
    {
        const quad X = a * d[0], Y = b * d[1], Z = c * d[2];
        switch (comp) {
        case 0: return F2(X, Y, Z);
        case 1: return F2(Y, X, Z);
        case 2: return F2(Z, Y, X);
        case 3: return G2(X, Y, Z);
        case 4: return G2(X, Z, Y);
        default: return G2(Y, Z, X);
        }
    }
};

} // namespace

// box[3]: number of offsets per axis (0..box_d-1) to fill; out[6][box2][box1][box0] (x fastest).
extern "C" int nm_newell_near_box(const int *box, const double *dx, double *out, int n_threads)
{
    const long b0 = box[0], b1 = box[1], b2 = box[2];
    if (b0 <= 0 || b1 <= 0 || b2 <= 0) return 0;
    const quad d0 = dx[0], d1 = dx[1], d2 = dx[2];
    const quad pref = -1 / (4 * M_PIq * d0 * d1 * d2);
    if (n_threads <= 0) n_threads = (int)std::max(1u, std::thread::hardware_concurrency());
    const long n_slabs = 6 * b2;
    n_threads = (int)std::min<long>(n_threads, n_slabs);
    std::atomic<long> next(0);
    auto worker = [&]() {
        // per slab (component, z offset): antiderivative on the three z planes c-1, c, c+1
        std::vector<quad> plane((size_t)3 * (b1 + 2) * (b0 + 2));
        for (;;) {
            const long s = next.fetch_add(1);
            if (s >= n_slabs) break;
            const int comp = (int)(s / b2);
            const long c = s % b2;
            Gen gen{comp, {d0, d1, d2}};
            for (int k = 0; k < 3; ++k)
                for (long b = -1; b <= b1; ++b)
                    for (long a = -1; a <= b0; ++a)
                        plane[((size_t)k * (b1 + 2) + (b + 1)) * (b0 + 2) + (a + 1)] =
                            gen(a, b, c + k - 1);
            static const int w3[3] = {1, -2, 1};
            for (long b = 0; b < b1; ++b)
                for (long a = 0; a < b0; ++a) {
                    quad sum = 0;
                    for (int k = 0; k < 3; ++k)
                        for (int j = 0; j < 3; ++j)
                            for (int i = 0; i < 3; ++i)
                                sum += (quad)(w3[i] * w3[j] * w3[k]) *
                                       plane[((size_t)k * (b1 + 2) + (b + j)) * (b0 + 2) + (a + i)];
                    out[(((size_t)comp * b2 + c) * b1 + b) * b0 + a] = (double)(pref * sum);
                }
        }
    };
    std::vector<std::thread> pool;
    for (int i = 1; i < n_threads; ++i) pool.emplace_back(worker);
    worker();
    for (auto &t : pool) t.join();
    return 0;
}
