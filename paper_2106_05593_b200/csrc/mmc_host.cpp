// mmc_host.cpp -- host-side set-up arithmetic of the MMC library (fp64 / binary128), no CUDA.
//  * thermal parameterisation: me(T) Eq. (9), chi(T) Eq. (8), longitudinal quartic of Eq. (7),
//    sigma of Eq. (13)
//  * demagnetising tensor of Eq. (14): Newell cell-averaged formulas in the near
//    field, evaluated in binary128 on a lattice of corner points followed by three 1-D second
//    differences; moment expansion of the point-dipole kernel in the far field.
// Written from the paper and the published Newell formulas; shares nothing with oracle/.
#include "mmc_internal.h"

#include <quadmath.h>

#include <algorithm>
#include <cmath>
#include <thread>
#include <vector>

namespace mmc {

// ---------------------------------------------------------------------------------------------
// Langevin function and the mean-field curve
// ---------------------------------------------------------------------------------------------
static double langevin(double x)
{
    // B(x) = coth x - 1/x.  Written as 1 + 2/expm1(2x) - 1/x for moderate x; the odd Taylor
    // polynomial below |x| < 0.25 where the two singular parts cancel.
    double ax = std::fabs(x);
    if (ax < 0.25) {
        double t = x * x;
        // x/3 - x^3/45 + 2x^5/945 - x^7/4725 + 2x^9/93555 - 1382x^11/638512875 + 4x^13/18243225
        double p = 4.0 / 18243225.0;
        p = p * t - 1382.0 / 638512875.0;
        p = p * t + 2.0 / 93555.0;
        p = p * t - 1.0 / 4725.0;
        p = p * t + 2.0 / 945.0;
        p = p * t - 1.0 / 45.0;
        p = p * t + 1.0 / 3.0;
        return p * x;
    }
    double s = x < 0 ? -1.0 : 1.0;
    double v = ax > 40.0 ? 1.0 - 1.0 / ax : 1.0 + 2.0 / std::expm1(2.0 * ax) - 1.0 / ax;
    return s * v;
}

static double langevin_deriv(double x)
{
    double ax = std::fabs(x);
    if (ax < 0.25) {
        double t = x * x;
        double p = 52.0 / 18243225.0;
        p = p * t - 15202.0 / 638512875.0;
        p = p * t + 18.0 / 93555.0;
        p = p * t - 7.0 / 4725.0;
        p = p * t + 10.0 / 945.0;
        p = p * t - 3.0 / 45.0;
        p = p * t + 1.0 / 3.0;
        return p;
    }
    if (ax > 300.0) return 1.0 / (x * x);
    double sh = std::sinh(ax);
    return 1.0 / (x * x) - 1.0 / (sh * sh);
}

// me = B(me * 3Tc/T) for T < Tc (Eq. (9) without the field term), solved in the variable
// x = me * a by a bracketed Newton iteration on h(x) = a B(x) - x.
static double solve_me(double T, double Tc)
{
    if (!(T < Tc)) return 0.0;
    const double a = 3.0 * Tc / T;
    double lo = 0.0, hi = a;                        // h(0+) > 0 (slope a/3 - 1 > 0), h(a) = a(B(a) - 1) < 0
    double x = std::min(a, std::sqrt(std::max(1e-300, 15.0 * (1.0 - 3.0 / a))));   // small-x estimate
    if (!(x > 0.0)) x = 0.5 * a;
    for (int it = 0; it < 200; ++it) {
        double h = a * langevin(x) - x;
        if (h > 0.0) lo = x; else hi = x;
        double dh = a * langevin_deriv(x) - 1.0;
        double xn = (dh != 0.0) ? x - h / dh : 0.5 * (lo + hi);
        if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
        if (std::fabs(xn - x) <= 4e-16 * std::fabs(xn)) { x = xn; break; }
        x = xn;
    }
    return x / a;
}

int thermal_coefficients(double T, double Tc, double mu, double V, double Ms0, ThermalCoef* o)
{
    if (!(T > 0.0) || !(Tc > 0.0) || !(mu > 0.0) || !(V > 0.0) || !(Ms0 > 0.0)) return MMC_E_INVALID;
    const double kT = kBoltzmann * T;
    ThermalCoef r{};
    if (std::fabs(T - Tc) < 1e-7 * Tc) {
        // common limit of both branches of Eq. (7): c2 -> 0, c4 -> (9/20) V Ms0 / mu
        r.me = 0.0; r.chi = INFINITY; r.c2 = 0.0; r.c4 = 0.45 * V * Ms0 / mu; r.mu2 = 0.0; r.sigma13 = 0.03;
    } else if (T < Tc) {
        r.me = solve_me(T, Tc);
        const double a = 3.0 * Tc / T;
        const double bp = langevin_deriv(r.me * a);
        r.chi = (mu / kT) * bp / (1.0 - bp * a);                       // Eq. (8)
        const double c = V * Ms0 / (8.0 * r.chi * r.me * r.me * kT);   // Eq. (7), T < Tc
        r.c4 = c; r.c2 = -2.0 * c * r.me * r.me; r.mu2 = r.me * r.me;
        r.sigma13 = std::min(0.03, 2.0 * r.me * std::sqrt(r.chi * kT / (V * Ms0)));   // Eq. (13) + cap
    } else {
        // Eq. (8) with me = 0: chi = mu / (3 kB (T - Tc)); Eq. (7), T > Tc
        r.me = 0.0;
        r.chi = mu / (3.0 * kBoltzmann * (T - Tc));
        r.c2 = V * Ms0 / (2.0 * r.chi * kT);
        r.c4 = r.c2 * 3.0 * Tc / (10.0 * (T - Tc));
        r.mu2 = -r.c2 / (2.0 * r.c4);
        r.sigma13 = 0.03;
    }
    *o = r;
    return MMC_OK;
}

// ---------------------------------------------------------------------------------------------
// Newell tensor, near field.  f is even in x, y, z; g is odd in x and y, even in z.
// asinh(p/q) is written ln((p + R)/q) with non-negative arguments.
// ---------------------------------------------------------------------------------------------
typedef __float128 quad;

static quad newell_f(quad x, quad y, quad z)
{
    x = fabsq(x); y = fabsq(y); z = fabsq(z);
    const quad xx = x * x, yy = y * y, zz = z * z;
    const quad R = sqrtq(xx + yy + zz);
    quad acc = (2 * xx - yy - zz) * R / 6;
    if (y > 0) { quad q = xx + zz; if (q > 0) acc += y * (zz - xx) * logq((y + R) / sqrtq(q)) / 2; }
    if (z > 0) { quad q = xx + yy; if (q > 0) acc += z * (yy - xx) * logq((z + R) / sqrtq(q)) / 2; }
    if (x > 0 && y > 0 && z > 0) acc -= x * y * z * atanq(y * z / (x * R));
    return acc;
}

static quad newell_g(quad x, quad y, quad z)
{
    quad sgn = 1;
    if (x < 0) { x = -x; sgn = -sgn; }
    if (y < 0) { y = -y; sgn = -sgn; }
    z = fabsq(z);
    if (x == 0 || y == 0) return 0;                       // every term carries a factor x*y or vanishes
    const quad xx = x * x, yy = y * y, zz = z * z;
    const quad R = sqrtq(xx + yy + zz);
    quad acc = -x * y * R / 3;
    acc += y * (3 * zz - yy) * logq((x + R) / sqrtq(yy + zz)) / 6;
    acc += x * (3 * zz - xx) * logq((y + R) / sqrtq(xx + zz)) / 6;
    if (z > 0) {
        acc += x * y * z * logq((z + R) / sqrtq(xx + yy));
        acc -= z * zz * atanq(x * y / (z * R)) / 6;
        acc -= z * yy * atanq(x * z / (y * R)) / 2;
        acc -= z * xx * atanq(y * z / (x * R)) / 2;
    }
    return sgn * acc;
}

// One tensor component on offsets [0,ex) x [0,ey) x [0,ez) (in cells of hx*hy*hz):
// lattice of function values on corner points -1..e, then the (-1, 2, -1) second difference along
// each axis in turn -- the 27-point sum of Newell's formula factorised.
static void near_component(quad (*fn)(quad, quad, quad), int ex, int ey, int ez, double hx, double hy, double hz,
                           std::vector<double>& out /* ex*ey*ez, x fastest */)
{
    const int lx = ex + 2, ly = ey + 2, lz = ez + 2;
    std::vector<quad> a((size_t)lx * ly * lz);
    auto at = [&](int i, int j, int k) -> quad& { return a[((size_t)k * ly + j) * lx + i]; };
    for (int k = 0; k < lz; ++k)
        for (int j = 0; j < ly; ++j)
            for (int i = 0; i < lx; ++i) at(i, j, k) = fn((quad)(i - 1) * hx, (quad)(j - 1) * hy, (quad)(k - 1) * hz);
    // second difference along x (result valid for i in 1..lx-2), stored back at i
    for (int k = 0; k < lz; ++k) for (int j = 0; j < ly; ++j) {
        quad prev = at(0, j, k);
        for (int i = 1; i < lx - 1; ++i) { quad cur = at(i, j, k); at(i, j, k) = 2 * cur - prev - at(i + 1, j, k); prev = cur; }
    }
    for (int k = 0; k < lz; ++k) for (int i = 1; i < lx - 1; ++i) {
        quad prev = at(i, 0, k);
        for (int j = 1; j < ly - 1; ++j) { quad cur = at(i, j, k); at(i, j, k) = 2 * cur - prev - at(i, j + 1, k); prev = cur; }
    }
    for (int j = 1; j < ly - 1; ++j) for (int i = 1; i < lx - 1; ++i) {
        quad prev = at(i, j, 0);
        for (int k = 1; k < lz - 1; ++k) { quad cur = at(i, j, k); at(i, j, k) = 2 * cur - prev - at(i, j, k + 1); prev = cur; }
    }
    const quad norm = 1 / (4 * M_PIq * (quad)hx * hy * hz);
    out.resize((size_t)ex * ey * ez);
    for (int k = 0; k < ez; ++k) for (int j = 0; j < ey; ++j) for (int i = 0; i < ex; ++i)
        out[((size_t)k * ey + j) * ex + i] = (double)(norm * at(i + 1, j + 1, k + 1));
}

// component q of {xx,yy,zz,xy,xz,yz} = f or g with permuted arguments
static void near_field(int q, int ex, int ey, int ez, double dx, double dy, double dz, std::vector<double>& out)
{
    std::vector<double> t;
    auto permuted = [&](quad (*fn)(quad, quad, quad), int p0, int p1, int p2) {
        // evaluate fn(u_{p0}, u_{p1}, u_{p2}) where u = (x,y,z): build on the permuted lattice, then un-permute
        const int e[3] = { ex, ey, ez }; const double h[3] = { dx, dy, dz };
        near_component(fn, e[p0], e[p1], e[p2], h[p0], h[p1], h[p2], t);
        out.resize((size_t)ex * ey * ez);
        int o[3];
        for (o[2] = 0; o[2] < ez; ++o[2]) for (o[1] = 0; o[1] < ey; ++o[1]) for (o[0] = 0; o[0] < ex; ++o[0])
            out[((size_t)o[2] * ey + o[1]) * ex + o[0]] = t[((size_t)o[p2] * e[p1] + o[p1]) * e[p0] + o[p0]];
    };
    switch (q) {
        case 0: permuted(newell_f, 0, 1, 2); break;   // N_xx: f(x,y,z)
        case 1: permuted(newell_f, 1, 0, 2); break;   // N_yy: f(y,x,z)
        case 2: permuted(newell_f, 2, 1, 0); break;   // N_zz: f(z,y,x)
        case 3: permuted(newell_g, 0, 1, 2); break;   // N_xy: g(x,y,z)
        case 4: permuted(newell_g, 0, 2, 1); break;   // N_xz: g(x,z,y)
        default: permuted(newell_g, 1, 2, 0); break;  // N_yz: g(y,z,x)
    }
}

// ---------------------------------------------------------------------------------------------
// Far field: N_ab(R) = V < K_ab(R + w) >, K_ab = (1/4 pi)(delta_ab/r^3 - 3 r_a r_b/r^5), w = u - v with u, v
// uniform in the cell => <w_c^2> = d_c^2/6.  Taylor to second order (the kernel is harmonic, so the
// correction vanishes for cubes):  N_ab = V [ K_ab + (1/12) sum_c d_c^2 d^2 K_ab/dx_c^2 ],
// d^4(1/r)/dx_a dx_b dx_c^2 = [105 x_a x_b x_c^2 - 15 r^2 (x_a x_b + x_c^2 d_ab + 2 x_a x_c d_bc + 2 x_b x_c d_ac)
//                              + 3 r^4 (d_ab + 2 d_ac d_bc)] / r^9 ,  K_ab = -(1/4 pi) d^2(1/r)/dx_a dx_b.
// ---------------------------------------------------------------------------------------------
static void far_field(double X, double Y, double Z, double dx, double dy, double dz, double out[6])
{
    const double x[3] = { X, Y, Z }, d2[3] = { dx * dx, dy * dy, dz * dz };
    const double r2 = X * X + Y * Y + Z * Z, r = std::sqrt(r2);
    const double ir3 = 1.0 / (r2 * r), ir5 = ir3 / r2, ir9 = ir5 / (r2 * r2);
    const double V = dx * dy * dz, pref = V / (4.0 * M_PI);
    static const int A[6] = { 0, 1, 2, 0, 0, 1 }, B[6] = { 0, 1, 2, 1, 2, 2 };
    for (int q = 0; q < 6; ++q) {
        const int a = A[q], b = B[q];
        const double dab = (a == b) ? 1.0 : 0.0;
        double K = dab * ir3 - 3.0 * x[a] * x[b] * ir5;
        double corr = 0.0;
        for (int c = 0; c < 3; ++c) {
            const double dac = (a == c) ? 1.0 : 0.0, dbc = (b == c) ? 1.0 : 0.0;
            const double t4 = (105.0 * x[a] * x[b] * x[c] * x[c]
                               - 15.0 * r2 * (x[a] * x[b] + x[c] * x[c] * dab + 2.0 * x[a] * x[c] * dbc + 2.0 * x[b] * x[c] * dac)
                               + 3.0 * r2 * r2 * (dab + 2.0 * dac * dbc)) * ir9;
            corr += d2[c] * (-t4);
        }
        out[q] = pref * (K + corr / 12.0);
    }
}

int demag_tensor_at(double dx, double dy, double dz, int ox, int oy, int oz, int r_near, double out[6])
{
    if (!(dx > 0 && dy > 0 && dz > 0)) return MMC_E_INVALID;
    const int aox = std::abs(ox), aoy = std::abs(oy), aoz = std::abs(oz);
    if (std::max(aox, std::max(aoy, aoz)) > r_near) {
        far_field(ox * dx, oy * dy, oz * dz, dx, dy, dz, out);
        return MMC_OK;
    }
    const double sx = ox < 0 ? -1 : 1, sy = oy < 0 ? -1 : 1, sz = oz < 0 ? -1 : 1;
    const double sg[6] = { 1, 1, 1, sx * sy, sx * sz, sy * sz };
    for (int q = 0; q < 6; ++q) {
        std::vector<double> t;
        near_field(q, aox + 1, aoy + 1, aoz + 1, dx, dy, dz, t);
        out[q] = sg[q] * t.back();
    }
    return MMC_OK;
}

// Octant table out[q][(oz*ny + oy)*nx + ox] for offsets >= 0.
void demag_tensor_octant(int nx, int ny, int nz, double dx, double dy, double dz, int r_near, std::vector<double> out[6])
{
    const size_t P = (size_t)nx * ny * nz;
    for (int q = 0; q < 6; ++q) out[q].assign(P, 0.0);
    const int ex = std::min(nx, r_near + 1), ey = std::min(ny, r_near + 1), ez = std::min(nz, r_near + 1);
    {
        std::vector<std::thread> th;
        std::vector<double> nf[6];
        for (int q = 0; q < 6; ++q) th.emplace_back([&, q] { near_field(q, ex, ey, ez, dx, dy, dz, nf[q]); });
        for (auto& t : th) t.join();
        for (int q = 0; q < 6; ++q)
            for (int k = 0; k < ez; ++k) for (int j = 0; j < ey; ++j) for (int i = 0; i < ex; ++i)
                out[q][((size_t)k * ny + j) * nx + i] = nf[q][((size_t)k * ey + j) * ex + i];
    }
    const unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    std::vector<std::thread> th;
    const size_t rows = (size_t)ny * nz;
    for (unsigned t = 0; t < nt; ++t)
        th.emplace_back([&, t] {
            for (size_t row = t; row < rows; row += nt) {
                const int oy = (int)(row % ny), oz = (int)(row / ny);
                for (int ox = 0; ox < nx; ++ox) {
                    if (ox < ex && oy < ey && oz < ez) continue;
                    double v[6];
                    far_field(ox * dx, oy * dy, oz * dz, dx, dy, dz, v);
                    for (int q = 0; q < 6; ++q) out[q][row * nx + ox] = v[q];
                }
            }
        });
    for (auto& t : th) t.join();
}

}  // namespace mmc
