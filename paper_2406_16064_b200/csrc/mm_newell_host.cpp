// mm_newell_host.cpp — near-field demag tensor for mm_init_demag (setup, once).
//
// Within a small box of offsets around the origin the cell-averaged tensor is evaluated from the
// closed forms of ref [20] of the paper (formulas restated in DESIGN.md R1) in
// __float128, because in fp64 they lose ~eps*R^3 to cancellation.  Outside the box the library
// integrates the defining dipole integral by Gauss-Legendre quadrature on the device
// (mm_lib.cu: tensor_far_kernel).  Compiled by g++ (nvcc's front end is not asked to parse
// __float128); linked into libmm.so.
#include <quadmath.h>
#include <cstdlib>
#include <thread>
#include <vector>

namespace {
typedef __float128 Q;

// F(x,y,z): the function whose 27-point second-difference stencil gives N_xx.  Even in x, y, z.
Q Ffun(Q x, Q y, Q z)
{
    x = fabsq(x); y = fabsq(y); z = fabsq(z);
    const Q xx = x * x, yy = y * y, zz = z * z, R = sqrtq(xx + yy + zz);
    Q acc = (2 * xx - yy - zz) * R / 6;
    if (x > 0 && y > 0 && z > 0) acc -= x * y * z * atanq(y * z / (x * R));
    if (y > 0 && xx + zz > 0) acc += y * (zz - xx) / 2 * asinhq(y / sqrtq(xx + zz));
    if (z > 0 && xx + yy > 0) acc += z * (yy - xx) / 2 * asinhq(z / sqrtq(xx + yy));
    return acc;
}

// G(x,y,z): same for N_xy.  Odd in x and y, even in z; called with x,y,z >= 0, sign applied by caller.
Q Gfun(Q x, Q y, Q z)
{
    const Q xx = x * x, yy = y * y, zz = z * z, R = sqrtq(xx + yy + zz);
    if (!(x > 0) || !(y > 0)) return 0;
    Q acc = -x * y * R / 3;
    acc += y * (3 * zz - yy) / 6 * asinhq(x / sqrtq(yy + zz));
    acc += x * (3 * zz - xx) / 6 * asinhq(y / sqrtq(xx + zz));
    if (z > 0) {
        acc += x * y * z * asinhq(z / sqrtq(xx + yy));
        acc -= z * zz / 6 * atanq(x * y / (z * R));
        acc -= z * yy / 2 * atanq(x * z / (y * R));
        acc -= z * xx / 2 * atanq(y * z / (x * R));
    }
    return acc;
}
}  // namespace

// out[comp][k][j][i] for 0 <= i < bx, 0 <= j < by, 0 <= k < bz; comp = xx,yy,zz,xy,xz,yz.
extern "C" void mm_newell_near_box(int bx, int by, int bz, double dx, double dy, double dz, double* out)
{
    const int gx = bx + 1, gy = by + 1, gz = bz + 1;
    const size_t Gn = (size_t)gx * gy * gz, Bn = (size_t)bx * by * bz;
    std::vector<Q> tab(Gn);
    const Q pref = 1 / (4 * M_PIq * (Q)dx * (Q)dy * (Q)dz);
    const int wgt[3] = { -1, 2, -1 };
    unsigned nthr = std::thread::hardware_concurrency();
    if (nthr == 0) nthr = 1;
    if (nthr > 16) nthr = 16;
    for (int comp = 0; comp < 6; comp++) {
        auto fill = [&](unsigned t) {
            for (size_t idx = t; idx < Gn; idx += nthr) {
                const int i = (int)(idx % gx), j = (int)((idx / gx) % gy), k = (int)(idx / ((size_t)gx * gy));
                const Q x = i * (Q)dx, y = j * (Q)dy, z = k * (Q)dz;
                Q v;
                switch (comp) {
                case 0: v = Ffun(x, y, z); break;
                case 1: v = Ffun(y, x, z); break;
                case 2: v = Ffun(z, y, x); break;
                case 3: v = Gfun(x, y, z); break;
                case 4: v = Gfun(x, z, y); break;
                default: v = Gfun(y, z, x); break;
                }
                tab[idx] = v;
            }
        };
        std::vector<std::thread> th;
        for (unsigned t = 0; t < nthr; t++) th.emplace_back(fill, t);
        for (auto& t : th) t.join();
        const bool ox = (comp == 3 || comp == 4), oy = (comp == 3 || comp == 5), oz = (comp == 4 || comp == 5);
        for (int k = 0; k < bz; k++)
            for (int j = 0; j < by; j++)
                for (int i = 0; i < bx; i++) {
                    Q sum = 0;
                    for (int p = -1; p <= 1; p++)
                        for (int q = -1; q <= 1; q++)
                            for (int r = -1; r <= 1; r++) {
                                int a = i + p, b = j + q, c = k + r, sg = wgt[p + 1] * wgt[q + 1] * wgt[r + 1];
                                if (a < 0) { a = -a; if (ox) sg = -sg; }
                                if (b < 0) { b = -b; if (oy) sg = -sg; }
                                if (c < 0) { c = -c; if (oz) sg = -sg; }
                                sum += (Q)sg * tab[a + (size_t)gx * (b + (size_t)gy * c)];
                            }
                    out[comp * Bn + i + (size_t)bx * (j + (size_t)by * k)] = (double)(sum * pref);
                }
    }
}
