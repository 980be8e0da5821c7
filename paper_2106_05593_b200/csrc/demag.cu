// demag.cu -- demagnetising field of Eq. (14): B_d = -mu0 N (*) M by zero-padded FFT convolution,
// with hand-written FFTs that never touch the padding.
//
//   kernel A  "rows"    S0+S1: for a tile of 4 mesh rows (all nz layers): M = Ms0 m straight from the colour-split
//                       state (even cells = real part, odd cells = imaginary part: the colour planes ARE the even/odd
//                       packing of the half-length real-FFT trick), FFT of length Px/2, untangle to the Px/2+1
//                       non-redundant frequencies, z-DFT across the layers in registers, store transposed:
//                       T[c][kz][kx][j]  (j fastest, so that a column is contiguous for kernel B).
//   kernel B  "columns" S1+S2+S3: one CTA per (kx, kz): the three components' columns (ny complex each, the zero
//                       padding to Py only implied) -> forward FFT -> real symmetric 3x3 tensor multiply in the
//                       transform's own output order (the tensor spectrum is stored in that order) -> inverse FFT ->
//                       the ny kept rows back in place.
//   kernel C  "rows^-1" S3: mirror of A: inverse z-DFT in registers, re-tangle, inverse FFT of length Px/2, and the
//                       real/imaginary parts go straight to the even/odd cells of the colour-split B_d.
// Each kernel exists twice: the generic shared-memory variant described above (fft_smem.cuh, any length) and the
// register-resident variant (fft_reg.cuh: 16 points per thread, compile-time lengths 2^8 .. 2^12) that the paper-sized
// meshes use.  In the latter the rows kernels work layer by layer (several CTAs per SM instead of one holding all layers)
// and the z direction belongs to the columns kernel, in one of two ways:
//   layer-pair sum  (columns_lp_kernel; several layers, nz * Py/16 <= 512 threads and the shared memory fits): no z transform
//                   at all; the nz layers' columns are transformed once each way and combined per frequency with the 2-D
//                   tensor spectra of the nz layer offsets, in place in U;
//   z-DFT           (columns_fast_kernel; otherwise, and the one-layer PLANAR case): CTA (kx, kz) sums plane kz of a DFT of the
//                   shortest linear length 2 nz - 1 from the nz layers in its loader, and the inverse z-DFT is a streaming
//                   pass of its own (z_inverse_kernel).
// Padded lengths are powers of two >= 2n-1 (any mesh size works).  All normalisation and -mu0 are folded into the
// tensor spectrum, which is built once at set-up in fp64 (host Newell/moment table -> device placement -> cuFFT D2Z).
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>

#include "fft_reg.cuh"
#include "fft_reg8.cuh"
#include "fft_smem.cuh"
#include "mmc_internal.h"

namespace mmc {

using fft::Plan;

struct DemagPlan {
    Geometry g;
    int Px, Py, Pz, Hx, Cx;          // padded lengths, Hx = Px/2 (complex row FFT length), Cx = Hx+1 frequencies
    int lgPz;
    Plan px, py;                     // stage plans of the length-Hx and length-Py transforms
    int RJ;                          // rows per CTA in kernels A and C
    int RS;                          // shared-memory row stride (float2) in kernels A and C
    size_t smemA, smemB;
    int threadsA, threadsB;
    float2* twx = nullptr;           // exp(-2 pi i k / Px), k < Px
    float2* twy = nullptr;           // exp(-2 pi i k / Py), k < Py
    bool fastB = false;              // columns: register-resident transform (fft_reg.cuh), Py in 2^8 .. 2^12
    float2* twB1 = nullptr;          // its twiddle tables (fftr::Twiddles), 15 * Py/16 entries each
    float2* twB2 = nullptr;
    bool fastA = false;              // rows: register-resident per-layer kernels (Hx in 2^8 .. 2^11); needs fastB (z-DFT outside the rows kernels)
    float2* T = nullptr;             // [3][Pz][Cx][ny]
    float2* U = nullptr;             // fastA with nz > 1: [3][nz][Cx][ny], the layers before the z-DFT and after its inverse
    float* nhat[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };   // [Pz/2+1][Cx][Py], position order in y
    // layer-pair columns kernel (several layers, no z transform): U is transformed in place, T and nhat do not exist
    bool cols8 = false;              // several layers, Py in 2^10 .. 2^12: columns8_kernel (8 points per thread, fft_reg8.cuh)
    float2* tw8 = nullptr;           // its twiddle table (fftr8::Shape::NTW entries)
    bool planar_split = false;       // one layer, fewer than two columns CTAs per SM: in-plane pair and z component in separate CTAs
    bool lp = false;
    int lpG = 1;                     // kx per CTA
    float* nh2[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };    // [nz][Cx][Py]: 2-D spectra per layer offset dz
};

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { if (err) *err = std::string(#x) + ": " + cudaGetErrorString(e_); return MMC_E_CUDA; } } while (0)
#define CF(x) do { cufftResult r_ = (x); if (r_ != CUFFT_SUCCESS) { if (err) *err = std::string(#x) + ": cufft error " + std::to_string((int)r_); return MMC_E_CUDA; } } while (0)

static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
static int padded_pow2(int n, int at_least) { int p = at_least; while (p < 2 * n - 1) p <<= 1; return p; }

// ------------------------------------------------------------------------------------------------ set-up kernels
// place the octant table on the padded periodic grid: offset o_d (|o_d| < N_d) at index o_d mod P_d, zero elsewhere;
// diagonal components even, N_ab odd in coordinates a and b.
__global__ void place_kernel(int nx, int ny, int nz, int Px, int Py, int Pz, const double* __restrict__ oct, int sx, int sy, int sz,
                             double* __restrict__ full)
{
    const long long n = (long long)Px * Py * Pz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(t % Px); const long long r = t / Px; const int y = (int)(r % Py), z = (int)(r / Py);
        int ox = x < nx ? x : x - Px, oy = y < ny ? y : y - Py, oz = z < nz ? z : z - Pz;
        double v = 0.0;
        if (ox > -nx && oy > -ny && oz > -nz) {
            double s = 1.0;
            if (ox < 0) { ox = -ox; s *= sx; }
            if (oy < 0) { oy = -oy; s *= sy; }
            if (oz < 0) { oz = -oz; s *= sz; }
            v = s * oct[((long long)oz * ny + oy) * nx + ox];
        }
        full[t] = v;
    }
}
// spectrum (D2Z layout [kz][ky][kx <= Px/2]) -> nhat[kz <= Pz/2][kx][p], p = position of ky in the y transform's output
__global__ void permute_kernel(const double2* __restrict__ spec, float* __restrict__ out, int Cx, int Py, int Kz, Plan py, double scale,
                               int fast_lg, int imag = 0)
{
    const long long n = (long long)Kz * Cx * Py;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int p = (int)(t % Py); const long long r = t / Py; const int kx = (int)(r % Cx), kz = (int)(r / Cx);
        // fast path: slot e of thread tid sits at p = e * (Py/16) + tid
        // eight-point path: slot e of thread tid sits at p = e * (Py/8) + tid
        const int ky = fast_lg < 0 ? fftr8::freq_of_slot8(-fast_lg, p % (Py >> 3), p / (Py >> 3))
                     : fast_lg ? fftr::freq_of_slot(fast_lg, p % (Py >> 4), p / (Py >> 4)) : fft::freq_of_pos(py, p);
        const double2 z = spec[((long long)kz * Py + ky) * Cx + kx];
        out[t] = (float)(scale * (imag ? z.y : z.x));
    }
}
__global__ void twiddle_kernel(float2* tw, int P)
{
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < P; k += gridDim.x * blockDim.x) {
        double s, c;
        sincospi(-2.0 * (double)k / (double)P, &s, &c);
        tw[k] = make_float2((float)c, (float)s);
    }
}

static int blocks_for(long long n) { long long b = (n + 255) / 256; return (int)(b > 148 * 32 ? 148 * 32 : (b < 1 ? 1 : b)); }

// ------------------------------------------------------------------------------------------------ kernels A and C
struct RowArgs {
    Geometry g;
    int Hx, lgHx, Cx, lgPx, RJ, lgRJ, RS;
    Plan px;
    const float2* twx;
    const float* m[3]; const float* Ms0; float Ms0_u;     // kernel A input (colour-split)
    float* bd[3];                                         // kernel C output (colour-split)
    float2* T;                                            // [3][PZ][Cx][ny]
};

// kernel A: grid (ceil(ny/RJ), 3 components); dynamic smem = RJ * nz * RS float2
template <int PZ>
__global__ void __launch_bounds__(512) rows_fwd_kernel(const RowArgs a)
{
    pdl_enter();
    extern __shared__ float2 sm[];
    const Geometry g = a.g;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int c = blockIdx.y, j0 = blockIdx.x * a.RJ;
    const int nrows = a.RJ * g.nz, Hx = a.Hx, hxr = (g.nx + 1) >> 1;
    const float* __restrict__ mc = a.m[c];
    // S0: M = Ms0 m; even cells -> real part, odd cells -> imaginary part (z[n] = x[2n] + i x[2n+1]); zero padding
    for (int idx = tid; idx < (nrows << a.lgHx); idx += nt) {
        const int r = idx >> a.lgHx, n = idx & (Hx - 1);
        const int k = r >> a.lgRJ, j = j0 + (r & (a.RJ - 1));
        float2 v = make_float2(0.f, 0.f);
        if (j < g.ny && n < hxr) {
            const int row = k * g.ny + j, par = (j + k) & 1;
            const unsigned se = (unsigned)par * (unsigned)g.H + (unsigned)row * g.hx + n;
            const unsigned so = (unsigned)(1 - par) * (unsigned)g.H + (unsigned)row * g.hx + n;
            v.x = (a.Ms0 ? __ldg(a.Ms0 + se) : a.Ms0_u) * __ldg(mc + se);
            if (2 * n + 1 < g.nx) v.y = (a.Ms0 ? __ldg(a.Ms0 + so) : a.Ms0_u) * __ldg(mc + so);
        }
        sm[r * a.RS + fft::pad(n)] = v;
    }
    __syncthreads();
    fft::fft_forward(a.px, sm, nrows, a.RS, a.twx, a.lgPx, tid, nt);
    // untangle: Z (length Hx, digit-reversed) -> X'[k] = 2 X[k], k = 0..Hx, with X the length-Px spectrum of the real row
    for (int idx = tid; idx < (nrows << a.lgHx); idx += nt) {
        const int r = idx >> a.lgHx, k = idx & (Hx - 1);
        if (2 * k > Hx) continue;
        float2* base = sm + r * a.RS;
        if (k == 0) {
            const float2 z0 = base[0];
            base[0] = make_float2(2.f * (z0.x + z0.y), 0.f);
            base[fft::pad(Hx)] = make_float2(2.f * (z0.x - z0.y), 0.f);
        } else {
            const int k2 = Hx - k;
            const int pa = fft::pad(fft::pos_of_freq(a.px, k)), pb = fft::pad(fft::pos_of_freq(a.px, k2));
            const float2 A = base[pa], B = base[pb];                 // Z[k], Z[Hx-k]
            const float2 S = make_float2(A.x + B.x, A.y - B.y), D = make_float2(A.x - B.x, A.y + B.y);
            const float2 t = fft::cmul(__ldg(a.twx + k), D);         // w^k (Z[k] - conj Z[Hx-k])
            base[pa] = make_float2(S.x + t.y, S.y - t.x);
            if (k2 != k) base[pb] = make_float2(S.x - t.y, -S.y - t.x);
        }
    }
    __syncthreads();
    // z-DFT across the layers (registers) and transposed store: lanes run over the RJ rows fastest
    const int items = a.Cx << a.lgRJ;
    for (int idx = tid; idx < items; idx += nt) {
        const int jj = idx & (a.RJ - 1), kx = idx >> a.lgRJ, j = j0 + jj;
        const int pp = fft::pad(kx < Hx ? fft::pos_of_freq(a.px, kx) : Hx);
        float2 v[PZ];
#pragma unroll
        for (int k = 0; k < PZ; ++k) v[k] = (k < g.nz) ? sm[((k << a.lgRJ) + jj) * a.RS + pp] : make_float2(0.f, 0.f);
        fft::dif<PZ, false>(v);
        if (j < g.ny) {
#pragma unroll
            for (int kz = 0; kz < PZ; ++kz)
                a.T[((size_t)(c * PZ + kz) * a.Cx + kx) * g.ny + j] = v[fft::bitrev<PZ>(kz)];
        }
    }
}

// kernel C: the mirror of kernel A
template <int PZ>
__global__ void __launch_bounds__(512) rows_inv_kernel(const RowArgs a)
{
    pdl_enter();
    extern __shared__ float2 sm[];
    const Geometry g = a.g;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int c = blockIdx.y, j0 = blockIdx.x * a.RJ;
    const int nrows = a.RJ * g.nz, Hx = a.Hx, hxr = (g.nx + 1) >> 1;
    const int items = a.Cx << a.lgRJ;
    for (int idx = tid; idx < items; idx += nt) {
        const int jj = idx & (a.RJ - 1), kx = idx >> a.lgRJ, j = j0 + jj;
        const int pp = fft::pad(kx < Hx ? fft::pos_of_freq(a.px, kx) : Hx);
        float2 v[PZ];
#pragma unroll
        for (int kz = 0; kz < PZ; ++kz)
            v[fft::bitrev<PZ>(kz)] = (j < g.ny) ? a.T[((size_t)(c * PZ + kz) * a.Cx + kx) * g.ny + j] : make_float2(0.f, 0.f);
        fft::dit<PZ, true>(v);
#pragma unroll
        for (int k = 0; k < PZ; ++k) if (k < g.nz) sm[((k << a.lgRJ) + jj) * a.RS + pp] = v[k];
    }
    __syncthreads();
    // re-tangle: Y[k], k = 0..Hx  ->  Z'[k] = 2 (E[k] + i O[k]) in the digit-reversed slots of the length-Hx transform
    for (int idx = tid; idx < (nrows << a.lgHx); idx += nt) {
        const int r = idx >> a.lgHx, k = idx & (Hx - 1);
        if (2 * k > Hx) continue;
        float2* base = sm + r * a.RS;
        if (k == 0) {
            const float y0 = base[0].x, yh = base[fft::pad(Hx)].x;
            base[0] = make_float2(y0 + yh, y0 - yh);
        } else {
            const int k2 = Hx - k;
            const int pa = fft::pad(fft::pos_of_freq(a.px, k)), pb = fft::pad(fft::pos_of_freq(a.px, k2));
            const float2 A = base[pa], B = base[pb];                 // Y[k], Y[Hx-k]
            const float2 E = make_float2(A.x + B.x, A.y - B.y), D = make_float2(A.x - B.x, A.y + B.y);
            const float2 O = fft::cmulc(D, __ldg(a.twx + k));        // (Y[k] - conj Y[Hx-k]) conj(w^k)
            base[pa] = make_float2(E.x - O.y, E.y + O.x);
            if (k2 != k) base[pb] = make_float2(E.x + O.y, -E.y + O.x);
        }
    }
    __syncthreads();
    fft::fft_inverse(a.px, sm, nrows, a.RS, a.twx, a.lgPx, tid, nt);
    // real part -> even cells, imaginary part -> odd cells of the colour-split B_d
    for (int idx = tid; idx < (nrows << a.lgHx); idx += nt) {
        const int r = idx >> a.lgHx, n = idx & (Hx - 1);
        const int k = r >> a.lgRJ, j = j0 + (r & (a.RJ - 1));
        if (j < g.ny && n < hxr) {
            const float2 v = sm[r * a.RS + fft::pad(n)];
            const int row = k * g.ny + j, par = (j + k) & 1;
            a.bd[c][(unsigned)par * (unsigned)g.H + (unsigned)row * g.hx + n] = v.x;
            if (2 * n + 1 < g.nx) a.bd[c][(unsigned)(1 - par) * (unsigned)g.H + (unsigned)row * g.hx + n] = v.y;
        }
    }
}

// ------------------------------------------------------------------------------------------------ kernel B
struct ColArgs {
    int ny, Cx, Py, lgPy, Pz, BS;
    Plan py;
    const float2* twy;
    float2* T;
    const float* nhat[6];
};

// grid (Cx, Pz); dynamic smem = 3 * BS float2
template <bool THREE_D>
__global__ void __launch_bounds__(256) columns_kernel(const ColArgs a)
{
    pdl_enter();
    extern __shared__ float2 sm[];
    const int tid = threadIdx.x, nt = blockDim.x;
    const int kx = blockIdx.x, kz = blockIdx.y;
    const int Py = a.Py, ny = a.ny, BS = a.BS;
    float2* col[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) col[c] = a.T + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
    for (int idx = tid; idx < 3 * Py; idx += nt) {
        const int c = idx >> a.lgPy, j = idx & (Py - 1);
        sm[c * BS + fft::pad(j)] = (j < ny) ? col[c][j] : make_float2(0.f, 0.f);
    }
    __syncthreads();
    fft::fft_forward(a.py, sm, 3, BS, a.twy, a.lgPy, tid, nt);
    // S2: B^ = K^ M^, K^ = -mu0/(2 Px Py Pz) N^ real and symmetric; planes kz and Pz-kz share |K^| (xz, yz odd in kz)
    const int kzs = (2 * kz <= a.Pz) ? kz : a.Pz - kz;
    const float sg = (2 * kz <= a.Pz) ? 1.f : -1.f;
    const size_t nb = ((size_t)kzs * a.Cx + kx) * Py;
    for (int p = tid; p < Py; p += nt) {
        const int pp = fft::pad(p);
        const float2 u = sm[pp], v = sm[BS + pp], w = sm[2 * BS + pp];
        const float xx = __ldg(a.nhat[0] + nb + p), yy = __ldg(a.nhat[1] + nb + p), zz = __ldg(a.nhat[2] + nb + p), xy = __ldg(a.nhat[3] + nb + p);
        float2 ox, oy, oz;
        ox.x = xx * u.x + xy * v.x; ox.y = xx * u.y + xy * v.y;
        oy.x = xy * u.x + yy * v.x; oy.y = xy * u.y + yy * v.y;
        oz.x = zz * w.x;            oz.y = zz * w.y;
        if (THREE_D) {
            const float xz = sg * __ldg(a.nhat[4] + nb + p), yz = sg * __ldg(a.nhat[5] + nb + p);
            ox.x += xz * w.x; ox.y += xz * w.y;
            oy.x += yz * w.x; oy.y += yz * w.y;
            oz.x += xz * u.x + yz * v.x; oz.y += xz * u.y + yz * v.y;
        }
        sm[pp] = ox; sm[BS + pp] = oy; sm[2 * BS + pp] = oz;
    }
    __syncthreads();
    fft::fft_inverse(a.py, sm, 3, BS, a.twy, a.lgPy, tid, nt);
    for (int idx = tid; idx < 3 * Py; idx += nt) {
        const int c = idx >> a.lgPy, j = idx & (Py - 1);
        if (j < ny) col[c][j] = sm[c * BS + fft::pad(j)];
    }
}

// ------------------------------------------------------------------------------------------------ kernels A and C, register-resident
// The x direction with the length-Hx transform of fft_reg.cuh (Hx = 2^LGH, 8 <= LGH <= 11), one (component, layer) per
// CTA: the z direction lives in the columns kernel (layer-pair sum, or z-DFT in its loader), so these kernels have no coupling between layers and
// T[c][k][kx][j] holds nz planes per component.
// block (RJ = 4, T = Hx/16): threadIdx.x = row of the tile (fastest, so that the four rows' values of one frequency are
// one 32-byte sector of the transposed array), threadIdx.y = thread of the row's transform.
// Shared memory per row: the two exchange buffers, which the natural-order spectrum (padded index k + (k>>4), needed for
// the mirror-frequency access of the real-transform (un)tangling) reuses between barriers.  Row strides are = 4 (mod 16)
// elements, so that the four rows of a half-warp sit in different bank groups.
// grid (ceil(ny/4), 3 components * nz layers).
#ifndef MMC_ROWS_RJ11
#define MMC_ROWS_RJ11 4
#endif
#ifndef MMC_ROWS_RJ10
#define MMC_ROWS_RJ10 4
#endif
template <int LGH> struct RowShape {
    using S = fftr::Shape<LGH>;
    static constexpr int Hx = S::N, T = S::T;
    static constexpr int RJ = LGH >= 11 ? MMC_ROWS_RJ11 : (LGH == 10 ? MMC_ROWS_RJ10 : 4);   // mesh rows per CTA
    static constexpr int CP = Hx + Hx / 16;              // pad(k) + pad(Hx - k) (+1 when k & 15 != 0); = pad(Hx)
    static constexpr int ES = (S::SMEM > CP ? S::SMEM : CP) + 16 / RJ;   // row stride: RJ rows of a half-warp in different bank groups
};
struct RowFastArgs {
    Geometry g;
    int Cx;
    float2 cu[16];                                        // exp(-2 pi i kconst(e) / Px): slot part of the (un)tangling root
    const float* m[3]; const float* Ms0; float Ms0_u;
    float* bd[3];
    float2* T;
};

template <int LGH>
__global__ void __launch_bounds__(RowShape<LGH>::RJ * RowShape<LGH>::T, RowShape<LGH>::RJ * RowShape<LGH>::T > 256 ? 1 : 2) rows_fwd_fast_kernel(const RowFastArgs a)
{
    pdl_enter();
    using R = RowShape<LGH>;
    constexpr int T = R::T, Hx = R::Hx;
    extern __shared__ float2 sm[];
    const Geometry g = a.g;
    const int nz = g.nz, ny = g.ny;
    const int jj = threadIdx.x, t = threadIdx.y;
    const int c = blockIdx.y / nz, k = blockIdx.y - c * nz, j = blockIdx.x * R::RJ + jj;
    const bool valid = j < ny;
    const int hxr = (g.nx + 1) >> 1;
    float2* s1 = sm + jj * R::ES;
    float2* s2 = s1 + R::S::S1;
    float2* nat = s1;
    const int pb = fftr::pbase<LGH>(t), kb = fftr::kbase<LGH>(t);
    const fftr::Twiddles tw{ fftr::root(t, Hx), fftr::root(t >> 4, T), nullptr, nullptr };
    const float* __restrict__ mc = a.m[c];
    // S0: M = Ms0 m; even cells -> real part, odd cells -> imaginary part; only n < Hx/2 can be non-zero
    float2 v[16];
    {
        const int row = k * ny + (valid ? j : 0), par = ((valid ? j : 0) + k) & 1;
        const unsigned be = (unsigned)par * (unsigned)g.H + (unsigned)row * g.hx;
        const unsigned bo = (unsigned)(1 - par) * (unsigned)g.H + (unsigned)row * g.hx;
        float2 raw[8], rws[8];
#pragma unroll
        for (int n1 = 0; n1 < 8; ++n1) {
            const int n = t + n1 * T;
            float2 x = make_float2(0.f, 0.f), ms = make_float2(a.Ms0_u, a.Ms0_u);
            if (valid && n < hxr) {
                x.x = __ldg(mc + be + n);
                if (a.Ms0) ms.x = __ldg(a.Ms0 + be + n);
                if (2 * n + 1 < g.nx) { x.y = __ldg(mc + bo + n); if (a.Ms0) ms.y = __ldg(a.Ms0 + bo + n); }
            }
            raw[n1] = x; rws[n1] = ms;
        }
#pragma unroll
        for (int n1 = 0; n1 < 8; ++n1) { v[n1] = make_float2(raw[n1].x * rws[n1].x, raw[n1].y * rws[n1].y); v[n1 + 8] = make_float2(0.f, 0.f); }
    }
    fftr::forward<LGH, true, false>(v, s1, s2, tw, t);
    if (R::S::R3 > 1) __syncthreads();                               // exchange buffer 2 is read (R3 == 1: forward ends with a barrier)
#pragma unroll
    for (int e = 0; e < 16; ++e) nat[pb + fftr::pconst<LGH>(e)] = v[e];
    __syncthreads();
    // untangle (X' = 2 X of the real row, from Z[k] and Z[Hx-k]) and transposed store
    const float2 wub = fftr::root(kb, 2 * Hx);
    float2* __restrict__ out = a.T + ((size_t)blockIdx.y * a.Cx) * ny + (valid ? j : 0);
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int kx = kb + fftr::kconst<LGH>(e);
        const int pa = pb + fftr::pconst<LGH>(e);
        const int pm = (kx == 0) ? pa : R::CP - pa - (fftr::lo_nonzero<LGH>(t, e) ? 1 : 0);
        const float2 w = fft::cmul(wub, a.cu[e]);
        const float2 A = v[e], B = nat[pm];
        const float2 Sm = make_float2(A.x + B.x, A.y - B.y), D = make_float2(A.x - B.x, A.y + B.y);
        const float2 tt = fft::cmul(w, D);
        if (valid) out[(size_t)kx * ny] = make_float2(Sm.x + tt.y, Sm.y - tt.x);
        if (e == 0 && t == 0 && valid) out[(size_t)Hx * ny] = make_float2(2.f * (A.x - A.y), 0.f);   // Nyquist column
    }
}

#ifndef MMC_ROWS_INV_MINB
#define MMC_ROWS_INV_MINB 2
#endif
template <int LGH>
__global__ void __launch_bounds__(RowShape<LGH>::RJ * RowShape<LGH>::T, RowShape<LGH>::RJ * RowShape<LGH>::T > 256 ? 1 : MMC_ROWS_INV_MINB) rows_inv_fast_kernel(const RowFastArgs a)
{
    pdl_enter();
    using R = RowShape<LGH>;
    constexpr int T = R::T, Hx = R::Hx;
    extern __shared__ float2 sm[];
    const Geometry g = a.g;
    const int nz = g.nz, ny = g.ny;
    const int jj = threadIdx.x, t = threadIdx.y;
    const int c = blockIdx.y / nz, k = blockIdx.y - c * nz, j = blockIdx.x * R::RJ + jj;
    const bool valid = j < ny;
    const int hxr = (g.nx + 1) >> 1;
    float2* s1 = sm + jj * R::ES;
    float2* s2 = s1 + R::S::S1;
    float2* nat = s1;
    const int pb = fftr::pbase<LGH>(t), kb = fftr::kbase<LGH>(t);
    const fftr::Twiddles tw{ fftr::root(t, Hx), fftr::root(t >> 4, T), nullptr, nullptr };
    const float2 wub = fftr::root(kb, 2 * Hx);
    const float2* __restrict__ in = a.T + ((size_t)blockIdx.y * a.Cx) * ny + (valid ? j : 0);
    float2 v[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = valid ? in[(size_t)(kb + fftr::kconst<LGH>(e)) * ny] : make_float2(0.f, 0.f);
    float2 yh = make_float2(0.f, 0.f);
    if (t == 0 && valid) yh = in[(size_t)Hx * ny];
#pragma unroll
    for (int e = 0; e < 16; ++e) nat[pb + fftr::pconst<LGH>(e)] = v[e];
    __syncthreads();
    // re-tangle: Y[k], Y[Hx-k] -> Z'[k] = 2 (E[k] + i O[k]) in this thread's slots
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int pa = pb + fftr::pconst<LGH>(e);
        const int pm = R::CP - pa - (fftr::lo_nonzero<LGH>(t, e) ? 1 : 0);
        const bool first = (e == 0 && t == 0);                     // k = 0: the mirror is the Nyquist value; both are real
        const float2 A = v[e], B = first ? yh : nat[first ? pa : pm];
        const float2 w = fft::cmul(wub, a.cu[e]);
        const float2 E = make_float2(A.x + B.x, A.y - B.y), D = make_float2(A.x - B.x, A.y + B.y);
        const float2 O = fft::cmulc(D, w);
        v[e] = first ? make_float2(A.x + B.x, A.x - B.x) : make_float2(E.x - O.y, E.y + O.x);
    }
    __syncthreads();                                                 // the natural-order array is read: exchanges may reuse it
    fftr::inverse<LGH, false>(v, s1, s2, tw, t);
    // real part -> even cells, imaginary part -> odd cells of the colour-split B_d
    float* __restrict__ bc = a.bd[c];
    const int row = k * ny + (valid ? j : 0), par = ((valid ? j : 0) + k) & 1;
    const unsigned be = (unsigned)par * (unsigned)g.H + (unsigned)row * g.hx;
    const unsigned bo = (unsigned)(1 - par) * (unsigned)g.H + (unsigned)row * g.hx;
#pragma unroll
    for (int n1 = 0; n1 < 8; ++n1) {
        const int n = t + n1 * T;
        if (valid && n < hxr) {
            bc[be + n] = v[n1].x;
            if (2 * n + 1 < g.nx) bc[bo + n] = v[n1].y;
        }
    }
}

template <int LGH>
static int launch_rows_fast(const DemagPlan* p, const RowFastArgs& ra, bool inverse, cudaStream_t st)
{
    using R = RowShape<LGH>;
    const dim3 grid((p->g.ny + R::RJ - 1) / R::RJ, 3 * p->g.nz), block(R::RJ, R::T);
    const size_t smem = (size_t)R::RJ * R::ES * sizeof(float2);
    if (inverse) {
        if (smem > 48 * 1024 && cudaFuncSetAttribute(rows_inv_fast_kernel<LGH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(rows_inv_fast_kernel<LGH>, dim3(grid), dim3(block), (size_t)(smem), st, ra);
    } else {
        if (smem > 48 * 1024 && cudaFuncSetAttribute(rows_fwd_fast_kernel<LGH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(rows_fwd_fast_kernel<LGH>, dim3(grid), dim3(block), (size_t)(smem), st, ra);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
static int launch_rows_fast_any(const DemagPlan* p, const RowFastArgs& ra, bool inverse, cudaStream_t st)
{
    switch (ilog2(p->Hx)) {
        case 8: return launch_rows_fast<8>(p, ra, inverse, st);
        case 9: return launch_rows_fast<9>(p, ra, inverse, st);
        case 10: return launch_rows_fast<10>(p, ra, inverse, st);
        case 11: return launch_rows_fast<11>(p, ra, inverse, st);
        default: return MMC_E_UNSUPPORTED;
    }
}

// kernel B, register-resident variant (fft_reg.cuh) for Py = 2^LGN, 8 <= LGN <= 12: T = Py/16 threads per (kx, kz)
// column set, G column sets (adjacent kx) per CTA.  Each thread keeps its 16 points of all three components in
// registers from the forward transform through the tensor multiply into the inverse transform; shared memory only
// carries the two exchanges of each transform.  HALF (2 ny == Py): the zero half of the input and the discarded half
// of the output are pruned at compile time.  grid (ceil(Cx/G), Pz), block (T, G).
struct ColFastArgs {
    int ny, Cx, Pz;
    int nz;                                    // > 0: forward z-DFT fused into the load: Tin holds nz layers per component
    const float2* tw1; const float2* tw2;      // fft_reg.cuh twiddle tables of the length-Py transform
    const float2* Tin;                         // [3][nz or Pz][Cx][ny]
    float2* Tout;                              // [3][Pz][Cx][ny] (== Tin when nz == 0: in place)
    const float* nhat[6];
};

#ifndef MMC_COLS_MINB
#define MMC_COLS_MINB 3
#endif
#ifndef MMC_COLS_MINB_PLANAR
#define MMC_COLS_MINB_PLANAR 3
#endif
#ifndef MMC_COLS_MINB_PLANAR_T256
#define MMC_COLS_MINB_PLANAR_T256 2
#endif
// PLANAR (one layer, Pz == 1, no xz / yz spectrum): B_z = K_zz M_z decouples from (B_x, B_y), so the in-plane pair and the
// z component go through the transforms one after the other and a thread holds two components instead of three.
template <int LGN, bool HALF, bool PLANAR>
__global__ void __launch_bounds__(fftr::Shape<LGN>::T * fftr::Shape<LGN>::G,
                                  fftr::Shape<LGN>::T >= 256 ? (PLANAR ? MMC_COLS_MINB_PLANAR_T256 : 2) : (PLANAR ? MMC_COLS_MINB_PLANAR : MMC_COLS_MINB))
columns_fast_kernel(const ColFastArgs a)
{
    pdl_enter();
    using S = fftr::Shape<LGN>;
    constexpr int N = S::N, T = S::T, NL = HALF ? 8 : 16;
    extern __shared__ float2 sm[];
    float2* s1 = sm + threadIdx.y * S::SMEM;
    float2* s2 = s1 + S::S1;
    const int tid = threadIdx.x;
    if constexpr (PLANAR) {
        const int kxr = blockIdx.x * S::G + threadIdx.y;
        const bool live = kxr < a.Cx;
        const int kx = live ? kxr : a.Cx - 1;
        const int ny = a.ny;
        const fftr::Twiddles tw{ make_float2(1.f, 0.f), make_float2(1.f, 0.f), a.tw1, a.tw2 };
        const size_t nb = (size_t)kx * N + tid;
        float2 v[2][16];
        // gridDim.y == 2 (small meshes, where the grid does not fill the GPU and the kernel's time is one warp's instruction
        // chain, not throughput): the in-plane pair and the z component, which share nothing, run in different CTAs
        const bool do_pair = gridDim.y == 1 || blockIdx.y == 0, do_z = gridDim.y == 1 || blockIdx.y == 1;
        // in-plane pair: load, the xx / yy / xy spectrum into L2 meanwhile, two forward transforms, 2x2 multiply, two inverse
        if (do_pair) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float2* __restrict__ col = a.Tin + ((size_t)c * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const int j = tid + n1 * T;
                v[c][n1] = (n1 < NL && (HALF || j < ny)) ? col[j] : make_float2(0.f, 0.f);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
#pragma unroll
            for (int e = 0; e < 16; ++e) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.nhat[q] + nb + e * T));
        }
#pragma unroll
        for (int c = 0; c < 2; ++c) fftr::forward<LGN, HALF, true>(v[c], s1, s2, tw, tid);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 u = v[0][e], w1 = v[1][e];
            const float xx = __ldg(a.nhat[0] + nb + e * T), yy = __ldg(a.nhat[1] + nb + e * T), xy = __ldg(a.nhat[3] + nb + e * T);
            v[0][e].x = fmaf(xx, u.x, xy * w1.x); v[0][e].y = fmaf(xx, u.y, xy * w1.y);
            v[1][e].x = fmaf(xy, u.x, yy * w1.x); v[1][e].y = fmaf(xy, u.y, yy * w1.y);
        }
        __syncthreads();                               // every thread is done reading exchange buffer 2
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            fftr::inverse<LGN, true>(v[c], s1, s2, tw, tid);
            float2* __restrict__ col = a.Tout + ((size_t)c * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < NL; ++n1) {
                const int j = tid + n1 * T;
                if (live && (HALF || j < ny)) col[j] = v[c][n1];
            }
        }
        }
        // z component in the registers of the first
        if (do_z) {
            float2 (&z)[16] = v[0];
            const float2* __restrict__ cin = a.Tin + ((size_t)2 * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const int j = tid + n1 * T;
                z[n1] = (n1 < NL && (HALF || j < ny)) ? cin[j] : make_float2(0.f, 0.f);
            }
            __syncthreads();                           // the last inverse transform read exchange buffer 1
            fftr::forward<LGN, HALF, true>(z, s1, s2, tw, tid);
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float zz = __ldg(a.nhat[2] + nb + e * T);
                z[e].x *= zz; z[e].y *= zz;
            }
            __syncthreads();
            fftr::inverse<LGN, true>(z, s1, s2, tw, tid);
            float2* __restrict__ col = a.Tout + ((size_t)2 * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < NL; ++n1) {
                const int j = tid + n1 * T;
                if (live && (HALF || j < ny)) col[j] = z[n1];
            }
        }
        return;
    }
    // with the fused z-DFT the Pz CTAs of one kx read the same layers: kz is the fastest block index so that they run
    // together and all but the first find them in L2
    const bool zf = a.nz > 0;
    const int kz = zf ? blockIdx.x : blockIdx.y;
    const int kxr = (zf ? blockIdx.y : blockIdx.x) * S::G + threadIdx.y;
    const bool live = kxr < a.Cx;                      // idle groups still walk through the barriers
    const int kx = live ? kxr : a.Cx - 1;
    const int ny = a.ny;
#ifndef MMC_COLS_TWS
#define MMC_COLS_TWS 0
#endif
    // MMC_COLS_TWS (measured and dropped, kept as a build knob): against the instruction-fetch stalls that top this kernel's list once
    // the additions are packed (ncu: no_instruction 1.6 of 6.2 warp cycles per instruction, instruction-cache hit rate 69 %), the
    // rolled variant (MMC_COLS_ROLL) does fit the cache (hit rate 98.6 %, no_instruction gone) but then waits on the twiddle loads it
    // can no longer hoist across transforms (long_scoreboard 1.2 -> 3.3: 0.302 ms); with the tables in shared memory it comes to
    // 0.258 ms rolled and 0.261 ms unrolled, against 0.228 ms for the straight-line kernel with L1-served tables (cfg 4)
#if MMC_COLS_TWS
    // twiddle tables in shared memory, copied once per CTA (fft_reg.cuh TABLE = 2: fetched where they are used)
    constexpr int TW = 2;
    float2* tws1 = sm + S::G * S::SMEM;
    float2* tws2 = tws1 + 15 * T;
    for (int i = threadIdx.y * T + tid; i < 15 * T; i += S::G * T) { tws1[i] = __ldg(a.tw1 + i); tws2[i] = __ldg(a.tw2 + i); }
    __syncthreads();
    const fftr::Twiddles tw{ make_float2(1.f, 0.f), make_float2(1.f, 0.f), tws1, tws2 };
#else
    constexpr int TW = 1;
    const fftr::Twiddles tw{ make_float2(1.f, 0.f), make_float2(1.f, 0.f), a.tw1, a.tw2 };
#endif
    float2 v[3][16];
    // all three components' columns are requested at once, and the tensor spectrum this thread will need after the
    // forward transforms is pulled into L2 meanwhile (no registers held)
    if (zf) {
        // S1, z direction: plane kz of the length-Pz DFT over the nz layers, X[kz] = sum_k w^(k kz) x[k], w = exp(-2 pi i / Pz)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz) * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < NL; ++n1) {
                const int j = tid + n1 * T;
                v[c][n1] = (HALF || j < ny) ? col[j] : make_float2(0.f, 0.f);
            }
        }
        const float2 wz = fftr::root(kz, a.Pz);
        float2 wk = wz;
#ifndef MMC_COLS_ZPIPE
#define MMC_COLS_ZPIPE 1
#endif
        if constexpr (HALF && MMC_COLS_ZPIPE) {
            // the upper halves of the register arrays are free until the transforms start (they hold the implied zero padding):
            // they carry the NEXT layer's values, requested right after the previous layer's values of the same component have
            // been consumed, i.e. two components' worth of arithmetic ahead of their use
            if (a.nz > 1) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + 1) * a.Cx + kx) * ny;
#pragma unroll
                    for (int n1 = 0; n1 < 8; ++n1) v[c][8 + n1] = col[tid + n1 * T];
                }
            }
            for (int k = 1; k < a.nz; ++k) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
#pragma unroll
                    for (int n1 = 0; n1 < 8; ++n1) {
                        const float2 x = v[c][8 + n1];
                        v[c][n1].x = fmaf(wk.x, x.x, fmaf(-wk.y, x.y, v[c][n1].x));
                        v[c][n1].y = fmaf(wk.x, x.y, fmaf(wk.y, x.x, v[c][n1].y));
                    }
                    if (k + 1 < a.nz) {
                        const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + k + 1) * a.Cx + kx) * ny;
#pragma unroll
                        for (int n1 = 0; n1 < 8; ++n1) v[c][8 + n1] = col[tid + n1 * T];
                    }
                }
                wk = fft::cmul(wk, wz);
            }
        } else {
            for (int k = 1; k < a.nz; ++k) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + k) * a.Cx + kx) * ny;
#pragma unroll
                    for (int n1 = 0; n1 < NL; ++n1) {
                        const int j = tid + n1 * T;
                        if (j < ny) {
                            const float2 x = col[j];
                            v[c][n1].x = fmaf(wk.x, x.x, fmaf(-wk.y, x.y, v[c][n1].x));
                            v[c][n1].y = fmaf(wk.x, x.y, fmaf(wk.y, x.x, v[c][n1].y));
                        }
                    }
                }
                wk = fft::cmul(wk, wz);
            }
        }
    } else if (HALF) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float2* __restrict__ col = a.Tin + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < 8; ++n1) v[c][n1] = col[tid + n1 * T];
        }
    }
    {
        const int kzs = (2 * kz <= a.Pz) ? kz : a.Pz - kz;
        const size_t nb = ((size_t)kzs * a.Cx + kx) * N + tid;
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            if (a.nhat[q] == nullptr) continue;
#pragma unroll
            for (int e = 0; e < 16; ++e) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.nhat[q] + nb + e * T));
        }
    }
#ifndef MMC_COLS_ROLL
#define MMC_COLS_ROLL 0
#endif
    // MMC_COLS_ROOT2 (default on): the constant roots inside the radix-16 butterflies of the three-component transforms as packed
    // FMUL2 + FFMA2 (fft::mul_root<.., P2>; same bits).  cfg 4 columns 0.2341 -> 0.2278 ms, cfg 6 0.3047 -> 0.2980; the one-layer
    // PLANAR instantiation (128-register cap at Py = 4096) spills with it (cfg 5 0.1457 -> 0.1522 ms) and the rows kernels do not
    // change, so only this branch uses it
#ifndef MMC_COLS_ROOT2
#define MMC_COLS_ROOT2 1
#endif
    // MMC_COLS_ROLL (measured and dropped, kept as a build knob): one copy of each transform in the instruction stream (the loops
    // over the components are not unrolled, the three register arrays rotate instead), against the 14 % of the warp cycles that
    // the 79 KB straight-line version stalls on instruction fetch: cfg 4 columns 0.265 ms rolled against 0.242 ms straight
#if MMC_COLS_ROLL
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
        if (HALF) {
#pragma unroll
            for (int n1 = 8; n1 < 16; ++n1) v[0][n1] = make_float2(0.f, 0.f);
        } else if (!zf) {
            const float2* __restrict__ col = a.Tin + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const int j = tid + n1 * T;
                v[0][n1] = (j < ny) ? col[j] : make_float2(0.f, 0.f);
            }
        }
        fftr::forward<LGN, HALF, TW, fftr::BlockSync, MMC_COLS_ROOT2 != 0>(v[0], s1, s2, tw, tid);
#pragma unroll
        for (int e = 0; e < 16; ++e) { const float2 t0 = v[0][e]; v[0][e] = v[1][e]; v[1][e] = v[2][e]; v[2][e] = t0; }
    }
#else
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (HALF) {
#pragma unroll
            for (int n1 = 8; n1 < 16; ++n1) v[c][n1] = make_float2(0.f, 0.f);
        } else if (!zf) {
            const float2* __restrict__ col = a.Tin + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const int j = tid + n1 * T;
                v[c][n1] = (j < ny) ? col[j] : make_float2(0.f, 0.f);
            }
        }
        fftr::forward<LGN, HALF, TW, fftr::BlockSync, MMC_COLS_ROOT2 != 0>(v[c], s1, s2, tw, tid);
    }
#endif
    // MMC_COLS_NH_CS=1: the tensor spectrum, read once per convolution, as streaming (evict-first) loads so that it does not push the
    // layers, which the Pz CTAs of a kx re-read, out of L2.  Measured: cfg 6 (10 layers, Pz = 19) 0.314 -> 0.305 ms, cfg 4 (Pz = 7)
    // 0.240 -> 0.247 ms: off.
#ifndef MMC_COLS_NH_CS
#define MMC_COLS_NH_CS 0
#endif
#if MMC_COLS_NH_CS
#define NH_LD(p) __ldcs(p)
#else
#define NH_LD(p) __ldg(p)
#endif
    // S2: B^ = K^ M^ (see columns_kernel); slot e of thread tid reads the permuted spectrum at e*T + tid
    {
        const int kzs = (2 * kz <= a.Pz) ? kz : a.Pz - kz;
        const float sg = (2 * kz <= a.Pz) ? 1.f : -1.f;
        const size_t nb = ((size_t)kzs * a.Cx + kx) * N + tid;
        const bool three_d = a.nhat[4] != nullptr;
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 u = v[0][e], w1 = v[1][e], w = v[2][e];
            const float xx = NH_LD(a.nhat[0] + nb + e * T), yy = NH_LD(a.nhat[1] + nb + e * T),
                        zz = NH_LD(a.nhat[2] + nb + e * T), xy = NH_LD(a.nhat[3] + nb + e * T);
            float2 ox, oy, oz;
            ox.x = fmaf(xx, u.x, xy * w1.x); ox.y = fmaf(xx, u.y, xy * w1.y);
            oy.x = fmaf(xy, u.x, yy * w1.x); oy.y = fmaf(xy, u.y, yy * w1.y);
            oz.x = zz * w.x;                 oz.y = zz * w.y;
            if (three_d) {
                const float xz = sg * NH_LD(a.nhat[4] + nb + e * T), yz = sg * NH_LD(a.nhat[5] + nb + e * T);
                ox.x = fmaf(xz, w.x, ox.x); ox.y = fmaf(xz, w.y, ox.y);
                oy.x = fmaf(yz, w.x, oy.x); oy.y = fmaf(yz, w.y, oy.y);
                oz.x = fmaf(xz, u.x, fmaf(yz, w1.x, oz.x)); oz.y = fmaf(xz, u.y, fmaf(yz, w1.y, oz.y));
            }
            v[0][e] = ox; v[1][e] = oy; v[2][e] = oz;
        }
    }
#undef NH_LD
    __syncthreads();                                   // every thread is done reading exchange buffer 2
#if MMC_COLS_ROLL
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
        fftr::inverse<LGN, TW, fftr::BlockSync, MMC_COLS_ROOT2 != 0>(v[0], s1, s2, tw, tid);
        float2* __restrict__ col = a.Tout + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < NL; ++n1) {
            const int j = tid + n1 * T;
            if (live && (HALF || j < ny)) col[j] = v[0][n1];
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) { const float2 t0 = v[0][e]; v[0][e] = v[1][e]; v[1][e] = v[2][e]; v[2][e] = t0; }
    }
#else
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        fftr::inverse<LGN, TW, fftr::BlockSync, MMC_COLS_ROOT2 != 0>(v[c], s1, s2, tw, tid);
        float2* __restrict__ col = a.Tout + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < NL; ++n1) {
            const int j = tid + n1 * T;
            if (live && (HALF || j < ny)) col[j] = v[c][n1];
        }
    }
#endif
}

// kernel B, eight points per thread (fft_reg8.cuh), several layers: the z-DFT path of columns_fast_kernel with T = Py/8 threads per
// (kx, kz) column set and 48 data registers per thread instead of 96.  grid (Pz, Cx), block T.  ColFastArgs::tw1 is the
// fftr8 twiddle table; the tensor spectrum is stored in fftr8's slot order (slot e of thread tid at e*T + tid).
#ifndef MMC_COLS8_MINB
#define MMC_COLS8_MINB 2
#endif
template <int LGN, bool HALF>
__global__ void __launch_bounds__(fftr8::Shape<LGN>::T, fftr8::Shape<LGN>::T >= 512 ? 1 : MMC_COLS8_MINB)
columns8_kernel(const ColFastArgs a)
{
    pdl_enter();
    using S = fftr8::Shape<LGN>;
    constexpr int N = S::N, T = S::T, NL = HALF ? 4 : 8;
    extern __shared__ float2 sm[];
    float2* s1 = sm;
    float2* s2 = sm + S::BUF;
    const int tid = threadIdx.x;
    const int kz = blockIdx.x, kx = blockIdx.y;        // kz fastest: the Pz CTAs of one kx find the layers in L2
    const int ny = a.ny;
    const float2* __restrict__ tw = a.tw1;
    float2 v[3][8];
    // S1, z direction: plane kz of the length-Pz DFT over the nz layers, X[kz] = sum_k w^(k kz) x[k], w = exp(-2 pi i / Pz)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < NL; ++n1) {
            const int j = tid + n1 * T;
            v[c][n1] = (HALF || j < ny) ? col[j] : make_float2(0.f, 0.f);
        }
    }
    const float2 wz = fftr::root(kz, a.Pz);
    float2 wk = wz;
    if constexpr (HALF) {
        // the upper halves of the register arrays (the implied zero padding) carry the next layer's values, requested right
        // after the previous layer's values of the same component have been consumed
        if (a.nz > 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + 1) * a.Cx + kx) * ny;
#pragma unroll
                for (int n1 = 0; n1 < 4; ++n1) v[c][4 + n1] = col[tid + n1 * T];
            }
        }
        for (int k = 1; k < a.nz; ++k) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
#pragma unroll
                for (int n1 = 0; n1 < 4; ++n1) {
                    const float2 x = v[c][4 + n1];
                    v[c][n1].x = fmaf(wk.x, x.x, fmaf(-wk.y, x.y, v[c][n1].x));
                    v[c][n1].y = fmaf(wk.x, x.y, fmaf(wk.y, x.x, v[c][n1].y));
                }
                if (k + 1 < a.nz) {
                    const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + k + 1) * a.Cx + kx) * ny;
#pragma unroll
                    for (int n1 = 0; n1 < 4; ++n1) v[c][4 + n1] = col[tid + n1 * T];
                }
            }
            wk = fft::cmul(wk, wz);
        }
    } else {
        for (int k = 1; k < a.nz; ++k) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float2* __restrict__ col = a.Tin + ((size_t)(c * a.nz + k) * a.Cx + kx) * ny;
#pragma unroll
                for (int n1 = 0; n1 < 8; ++n1) {
                    const int j = tid + n1 * T;
                    if (j < ny) {
                        const float2 x = col[j];
                        v[c][n1].x = fmaf(wk.x, x.x, fmaf(-wk.y, x.y, v[c][n1].x));
                        v[c][n1].y = fmaf(wk.x, x.y, fmaf(wk.y, x.x, v[c][n1].y));
                    }
                }
            }
            wk = fft::cmul(wk, wz);
        }
    }
    const int kzs = (2 * kz <= a.Pz) ? kz : a.Pz - kz;
    const float sg = (2 * kz <= a.Pz) ? 1.f : -1.f;
    const size_t nb = ((size_t)kzs * a.Cx + kx) * N + tid;
#pragma unroll
    for (int q = 0; q < 6; ++q) {
#pragma unroll
        for (int e = 0; e < 8; ++e) asm volatile("prefetch.global.L2 [%0];" ::"l"(a.nhat[q] + nb + e * T));
    }
    fftr8::forward<LGN, HALF>(v[0], s1, s2, tw, tid);
    fftr8::forward<LGN, HALF>(v[1], s2, s1, tw, tid);
    fftr8::forward<LGN, HALF>(v[2], s1, s2, tw, tid);
    // S2: B^ = K^ M^ (see columns_kernel)
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        const float2 u = v[0][e], w1 = v[1][e], w = v[2][e];
        const float xx = __ldg(a.nhat[0] + nb + e * T), yy = __ldg(a.nhat[1] + nb + e * T), zz = __ldg(a.nhat[2] + nb + e * T),
                    xy = __ldg(a.nhat[3] + nb + e * T), xz = sg * __ldg(a.nhat[4] + nb + e * T), yz = sg * __ldg(a.nhat[5] + nb + e * T);
        float2 ox, oy, oz;
        ox.x = fmaf(xx, u.x, xy * w1.x); ox.y = fmaf(xx, u.y, xy * w1.y);
        oy.x = fmaf(xy, u.x, yy * w1.x); oy.y = fmaf(xy, u.y, yy * w1.y);
        oz.x = zz * w.x;                 oz.y = zz * w.y;
        ox.x = fmaf(xz, w.x, ox.x); ox.y = fmaf(xz, w.y, ox.y);
        oy.x = fmaf(yz, w.x, oy.x); oy.y = fmaf(yz, w.y, oy.y);
        oz.x = fmaf(xz, u.x, fmaf(yz, w1.x, oz.x)); oz.y = fmaf(xz, u.y, fmaf(yz, w1.y, oz.y));
        v[0][e] = ox; v[1][e] = oy; v[2][e] = oz;
    }
    __syncthreads();                                   // every thread is done reading the exchange buffers
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (c == 1) fftr8::inverse<LGN>(v[c], s2, s1, tw, tid);
        else        fftr8::inverse<LGN>(v[c], s1, s2, tw, tid);
        float2* __restrict__ col = a.Tout + ((size_t)(c * a.Pz + kz) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < NL; ++n1) {
            const int j = tid + n1 * T;
            if (HALF || j < ny) col[j] = v[c][n1];
        }
    }
}

// ------------------------------------------------------------------------------------------------ kernel B, layer-pair variant
// Several layers WITHOUT a z transform (Eq. (14), written out in z): in the 2-D Fourier domain of one layer
//     B^_k(kx, ky) = sum_k' K^(kx, ky; k - k') M^_k'(kx, ky),      K^(.; dz) = 2-D spectrum of -mu0 N(x, y, dz),
// so the nz layers' columns are transformed once each way (3 nz forward + 3 nz inverse transforms per kx instead of the
// 3 (2 nz - 1) + 3 (2 nz - 1) of a length-(2 nz - 1) z-DFT), the z direction costs nz^2 small 3x3 products per frequency, and
// neither the z planes nor the inverse z pass exist.  One CTA per kx (G of them for short transforms): thread group k
// (threadIdx.y, T = Py/16 threads) owns layer k: load its three columns, three forward transforms (registers, fft_reg.cuh),
// then the layers meet through shared memory in chunks of EC register slots (a slot is one frequency: the sum over layers
// and components for a chunk is complete within the chunk, so the result replaces the chunk in the same registers),
// three inverse transforms, store in place.  The exchange reuses the transforms' exchange buffers (double-buffered chunks).
// Tensor spectra: nh[q][dz][kx][slot], dz = 0 .. nz-1; diagonal and xy components are even in dz and real; xz and yz are odd
// in dz and (odd in one in-plane coordinate only) purely imaginary: nh[4], nh[5] hold the imaginary parts.
struct ColLPArgs {
    int ny, Cx;
    const float2* tw1; const float2* tw2;      // fft_reg.cuh twiddle tables of the length-Py transform
    float2* U;                                 // [3][nz][Cx][ny], transformed in place
    const float* nh[6];
};

template <int LGN> struct LPShape { static constexpr int EC = 2, NC = 16 / EC; };   // slots per chunk; 2 * 3 EC T <= Shape::SMEM
// planes of the tensor spectrum per chunk row: dz = 0 has 4 components (xz = yz = 0), every other dz has 6
__host__ __device__ constexpr int lp_planes(int nz) { return 4 + 6 * (nz - 1); }
__host__ __device__ constexpr int lp_plane_index(int d, int q) { return d == 0 ? q : 4 + 6 * (d - 1) + q; }

// Shared memory: [transform exchange buffers of the G * nz groups | the two twiddle tables | two chunks of tensor spectrum |
// two mbarriers]: ~210 KB for four layers of Py = 2048, so there is no L1 to speak of: the twiddle tables live in shared
// memory too (read where they are used: no 15-entry register staging), and the kernel must not spill (a CTA's spill
// footprint would be L2 traffic).
// The tensor spectrum of a chunk (EC consecutive slots = EC * T consecutive floats of each plane) is brought in by
// cp.async.bulk copies that complete on an mbarrier, two chunks ahead of their use: the first two are requested before the
// forward transforms start, chunk ch + 2 as soon as chunk ch has been consumed, so no thread ever waits for these loads.
template <int LGN, bool HALF>
__global__ void __launch_bounds__(512, 1) columns_lp_kernel(const ColLPArgs a)
{
    pdl_enter();
    using S = fftr::Shape<LGN>;
    constexpr int N = S::N, T = S::T, NL = HALF ? 8 : 16, EC = LPShape<LGN>::EC, NC = LPShape<LGN>::NC;
    extern __shared__ float2 sm[];
    const int tid = threadIdx.x, k = threadIdx.y, g = threadIdx.z, nz = blockDim.y, G = blockDim.z;
    const int grp = g * nz + k;
    float2* s1 = sm + grp * S::SMEM;
    float2* s2 = s1 + S::S1;
    const int NP = lp_planes(nz);
    float2* tws1 = sm + G * nz * S::SMEM;                                    // fft_reg.cuh twiddle tables, 15 T entries each
    float2* tws2 = tws1 + 15 * T;
    float* tens = reinterpret_cast<float*>(tws2 + 15 * T);                   // [2][G][NP][EC * T]
    const int tbuf = G * NP * EC * T;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(tens + 2 * tbuf);
    const int kxr = blockIdx.x * G + g;
    const bool live = kxr < a.Cx;                      // idle groups still walk through the barriers
    const int kx = live ? kxr : a.Cx - 1;
    const int ny = a.ny;
    const fftr::Twiddles tw{ make_float2(1.f, 0.f), make_float2(1.f, 0.f), tws1, tws2 };
    const size_t plane = (size_t)a.Cx * N;             // one dz plane of a tensor component
    if (tid == 0 && grp == 0) { fftr::mbar_init(bar, G * nz); fftr::mbar_init(bar + 1, G * nz); fftr::mbar_fence_init(); }
    for (int i = grp * T + tid; i < 15 * T; i += G * nz * T) { tws1[i] = __ldg(a.tw1 + i); tws2[i] = __ldg(a.tw2 + i); }
    __syncthreads();
    // thread 0 of group (g, k) requests plane dz = k of this kx for chunk ch: one copy of EC * T floats per component
    auto request = [&](int ch) {
        if (tid != 0) return;
        const int nq = k == 0 ? 4 : 6;
        unsigned long long* b = bar + (ch & 1);
        fftr::mbar_arrive_expect_tx(b, (unsigned)(nq * EC * T * sizeof(float)));
        float* dst = tens + (ch & 1) * tbuf + (g * NP + lp_plane_index(k, 0)) * (EC * T);
        for (int q = 0; q < nq; ++q)
            fftr::bulk_copy_g2s(dst + q * (EC * T), a.nh[q] + (size_t)k * plane + (size_t)kx * N + ch * (EC * T),
                                (unsigned)(EC * T * sizeof(float)), b);
    };
    request(0);
    request(1);
    float2 v[3][16];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float2* __restrict__ col = a.U + ((size_t)(c * nz + k) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const int j = tid + n1 * T;
            v[c][n1] = (n1 < NL && (HALF || j < ny)) ? col[j] : make_float2(0.f, 0.f);
        }
    }
    // transforms of different layers do not wait for one another: one named barrier per group (warp-aligned groups only)
    constexpr bool GROUPS = T >= 64;
    const fftr::GroupSync gsync{ 1 + grp, T };
    // ONE copy of each transform in the instruction stream: the loops below are not unrolled; instead the register arrays
    // rotate (component-wise here, chunk-wise in the multiply), so that the loop body always works on v[0] / the first EC
    // slots.  Straight-line code for all components and chunks is ~100 KB and starves the instruction cache (measured: 45 %
    // of the warp cycles stalled on instruction fetch); the rotations cost ~15 % more instructions.
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
        if constexpr (GROUPS) fftr::forward<LGN, HALF, 2>(v[0], s1, s2, tw, tid, gsync);
        else fftr::forward<LGN, HALF, 2>(v[0], s1, s2, tw, tid);
#pragma unroll
        for (int e = 0; e < 16; ++e) { const float2 t0 = v[0][e]; v[0][e] = v[1][e]; v[1][e] = v[2][e]; v[2][e] = t0; }
    }
    __syncthreads();                                   // every group is done with its exchange buffers: they now carry the layers
    // S2 with the z direction as a direct sum over layer pairs.  xb[buf][g][layer][component][slot of the chunk][tid]
    constexpr int XS = 3 * EC * T;                     // one layer of one chunk
    float2* xb = sm + g * nz * XS;
    const int xbuf = G * nz * XS;                      // one buffer (all groups)
    {
        float2* w = xb + k * XS + tid;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int e = 0; e < EC; ++e) w[(c * EC + e) * T] = v[c][e];
    }
    __syncthreads();
#pragma unroll 1
    for (int ch = 0; ch < NC; ++ch) {                  // the current chunk sits in slots 0 .. EC-1 (the slots rotate, see below)
        if (ch + 1 < NC) {                             // the next chunk goes to the other buffer while this one is consumed
            float2* w = xb + ((ch + 1) & 1) * xbuf + k * XS + tid;
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int e = 0; e < EC; ++e) w[(c * EC + e) * T] = v[c][EC + e];
        }
        fftr::mbar_wait(bar + (ch & 1), (ch >> 1) & 1);                     // this chunk's tensor spectrum has landed
        const float2* r = xb + (ch & 1) * xbuf + tid;
        const float* tc = tens + (ch & 1) * tbuf + g * NP * (EC * T) + tid;
#pragma unroll
        for (int e = 0; e < EC; ++e) {
            float2 ox = make_float2(0.f, 0.f), oy = ox, oz = ox;
#pragma unroll 1
            for (int d = 0; d < nz; ++d) {
                const float* t = tc + lp_plane_index(d, 0) * (EC * T) + e * T;
                const float xx = t[0], yy = t[EC * T], zz = t[2 * EC * T], xy = t[3 * EC * T];
                float xz = 0.f, yz = 0.f;
                if (d > 0) { xz = t[4 * EC * T]; yz = t[5 * EC * T]; }
                // layer k' = k - d (offset +d) and, for d > 0, k' = k + d (offset -d: xz, yz change sign)
#pragma unroll
                for (int side = 0; side < 2; ++side) {
                    const int kp = side ? k + d : k - d;
                    if (side ? (d == 0 || kp >= nz) : (kp < 0)) continue;
                    const float2* m = r + kp * XS + e * T;
                    const float2 mx = m[0], my = m[EC * T], mz = m[2 * EC * T];
                    const float sxz = side ? -xz : xz, syz = side ? -yz : yz;
                    // (i s)(p + i q) = -s q + i s p
                    ox.x = fmaf(xx, mx.x, fmaf(xy, my.x, fmaf(-sxz, mz.y, ox.x)));
                    ox.y = fmaf(xx, mx.y, fmaf(xy, my.y, fmaf(sxz, mz.x, ox.y)));
                    oy.x = fmaf(xy, mx.x, fmaf(yy, my.x, fmaf(-syz, mz.y, oy.x)));
                    oy.y = fmaf(xy, mx.y, fmaf(yy, my.y, fmaf(syz, mz.x, oy.y)));
                    oz.x = fmaf(-sxz, mx.y, fmaf(-syz, my.y, fmaf(zz, mz.x, oz.x)));
                    oz.y = fmaf(sxz, mx.x, fmaf(syz, my.x, fmaf(zz, mz.y, oz.y)));
                }
            }
            v[0][e] = ox; v[1][e] = oy; v[2][e] = oz;
        }
        __syncthreads();                               // chunk consumed by all layers; after the last one the buffers go back to the transforms
        if (ch + 2 < NC) request(ch + 2);              // its buffers are free again
#pragma unroll
        for (int c = 0; c < 3; ++c) {                  // rotate the slots by one chunk (NC rotations restore the order)
            float2 t0[EC];
#pragma unroll
            for (int e = 0; e < EC; ++e) t0[e] = v[c][e];
#pragma unroll
            for (int e = 0; e < 16 - EC; ++e) v[c][e] = v[c][e + EC];
#pragma unroll
            for (int e = 0; e < EC; ++e) v[c][16 - EC + e] = t0[e];
        }
    }
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
        if constexpr (GROUPS) fftr::inverse<LGN, 2>(v[0], s1, s2, tw, tid, gsync);
        else fftr::inverse<LGN, 2>(v[0], s1, s2, tw, tid);
        float2* __restrict__ col = a.U + ((size_t)(c * nz + k) * a.Cx + kx) * ny;
#pragma unroll
        for (int n1 = 0; n1 < NL; ++n1) {
            const int j = tid + n1 * T;
            if (live && (HALF || j < ny)) col[j] = v[0][n1];
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) { const float2 t0 = v[0][e]; v[0][e] = v[1][e]; v[1][e] = v[2][e]; v[2][e] = t0; }
    }
}

// S3, z direction, for the per-layer rows kernels: inverse length-Pz DFT (Pz = 2 NZ - 1, a direct sum) across the planes of
// every (component, kx, j), the NZ kept layers written to `out` [3][NZ][Cx][ny].  A plain streaming pass (reads 8 Pz,
// writes 8 NZ bytes per point).
constexpr int kMaxFastLayers = 16;
template <int NZ>
__global__ void __launch_bounds__(256) z_inverse_kernel(const float2* __restrict__ in, float2* __restrict__ out, size_t plane)
{
    pdl_enter();
    constexpr int PZ = 2 * NZ - 1;
    __shared__ float2 w[PZ];                               // exp(+2 pi i q / Pz)
    if (threadIdx.x < PZ) { const float2 r = fftr::root(threadIdx.x, PZ); w[threadIdx.x] = make_float2(r.x, -r.y); }
    __syncthreads();
#ifndef MMC_ZINV_REVERSE
#define MMC_ZINV_REVERSE 1
#endif
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < plane; i0 += (size_t)gridDim.x * blockDim.x) {
        // from the end of the planes backwards: the columns kernel wrote them in ascending kx, so their tail is what L2 still holds
        // (cfg 4: 45.8 -> 44.0 us, measured twice each way)
        const size_t i = MMC_ZINV_REVERSE ? plane - 1 - i0 : i0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float2 x[PZ];
#pragma unroll
            for (int kz = 0; kz < PZ; ++kz) x[kz] = __ldcs(in + (size_t)(c * PZ + kz) * plane + i);
#pragma unroll
            for (int k = 0; k < NZ; ++k) {
                float2 acc = x[0];
#pragma unroll
                for (int kz = 1; kz < PZ; ++kz) {
                    const float2 t = w[(k * kz) % PZ];
                    acc.x = fmaf(t.x, x[kz].x, fmaf(-t.y, x[kz].y, acc.x));
                    acc.y = fmaf(t.x, x[kz].y, fmaf(t.y, x[kz].x, acc.y));
                }
                out[(size_t)(c * NZ + k) * plane + i] = acc;
            }
        }
    }
}
static int launch_z_inverse(const DemagPlan* p, const float2* in, float2* out, cudaStream_t st)
{
    const size_t plane = (size_t)p->Cx * p->g.ny;
    const int blocks = (int)std::min<size_t>((plane + 255) / 256, (size_t)148 * 16);
    switch (p->g.nz) {
        case 2: launch_pdl(z_inverse_kernel<2>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 3: launch_pdl(z_inverse_kernel<3>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 4: launch_pdl(z_inverse_kernel<4>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 5: launch_pdl(z_inverse_kernel<5>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 6: launch_pdl(z_inverse_kernel<6>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 7: launch_pdl(z_inverse_kernel<7>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 8: launch_pdl(z_inverse_kernel<8>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 9: launch_pdl(z_inverse_kernel<9>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 10: launch_pdl(z_inverse_kernel<10>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 11: launch_pdl(z_inverse_kernel<11>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 12: launch_pdl(z_inverse_kernel<12>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 13: launch_pdl(z_inverse_kernel<13>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 14: launch_pdl(z_inverse_kernel<14>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 15: launch_pdl(z_inverse_kernel<15>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        case 16: launch_pdl(z_inverse_kernel<16>, dim3(blocks), dim3(256), (size_t)(0), st, in, out, plane); break;
        default: return MMC_E_UNSUPPORTED;
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

template <int LGN, bool HALF>
static int launch_columns_fast_h(const DemagPlan* p, const ColFastArgs& ca, cudaStream_t st)
{
    using S = fftr::Shape<LGN>;
    const size_t smem = (size_t)S::G * S::SMEM * sizeof(float2);
    const unsigned nbx = (p->Cx + S::G - 1) / S::G;
    if (ca.nz == 0 && p->Pz == 1 && ca.nhat[4] == nullptr && ca.nhat[5] == nullptr) {      // one layer: the planar variant
        auto kp = columns_fast_kernel<LGN, HALF, true>;
        if (smem > 48 * 1024 && cudaFuncSetAttribute(kp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(kp, dim3(nbx, p->planar_split ? 2 : 1), dim3(S::T, S::G), smem, st, ca);
        return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
    }
    auto kern = columns_fast_kernel<LGN, HALF, false>;
#if defined(MMC_COLS_TWS) && MMC_COLS_TWS
#define MMC_COLS_TWS_EXTRA ((size_t)2 * 15 * S::T * sizeof(float2))
#else
#define MMC_COLS_TWS_EXTRA ((size_t)0)
#endif
    if (smem + MMC_COLS_TWS_EXTRA > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(smem + MMC_COLS_TWS_EXTRA)) != cudaSuccess) return MMC_E_CUDA;
    const dim3 grid = ca.nz > 0 ? dim3(p->Pz, nbx) : dim3(nbx, p->Pz), block(S::T, S::G);
    if (grid.y > 65535u) return MMC_E_UNSUPPORTED;
    launch_pdl(kern, dim3(grid), dim3(block), (size_t)(smem + MMC_COLS_TWS_EXTRA), st, ca);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
template <int LGN>
static int launch_columns_fast(const DemagPlan* p, const ColFastArgs& ca, cudaStream_t st)
{
    return 2 * p->g.ny == p->Py ? launch_columns_fast_h<LGN, true>(p, ca, st) : launch_columns_fast_h<LGN, false>(p, ca, st);
}
template <int LGN>
static size_t lp_smem_bytes(int nz, int G)
{
    using S = fftr::Shape<LGN>;
    return (size_t)G * nz * S::SMEM * sizeof(float2) + (size_t)2 * 15 * S::T * sizeof(float2)
           + (size_t)2 * G * lp_planes(nz) * LPShape<LGN>::EC * S::T * sizeof(float) + 2 * sizeof(unsigned long long);
}
static size_t lp_smem_bytes_any(int lgN, int nz, int G)
{
    switch (lgN) {
        case 8: return lp_smem_bytes<8>(nz, G);
        case 9: return lp_smem_bytes<9>(nz, G);
        case 10: return lp_smem_bytes<10>(nz, G);
        case 11: return lp_smem_bytes<11>(nz, G);
        case 12: return lp_smem_bytes<12>(nz, G);
        default: return ~(size_t)0;
    }
}
template <int LGN>
static int launch_columns_lp(const DemagPlan* p, const ColLPArgs& la, cudaStream_t st)
{
    using S = fftr::Shape<LGN>;
    const int G = p->lpG, nz = p->g.nz;
    const size_t smem = lp_smem_bytes<LGN>(nz, G);
    if (smem > 227 * 1024) return MMC_E_UNSUPPORTED;
    const dim3 grid((p->Cx + G - 1) / G), block(S::T, nz, G);
    if (2 * p->g.ny == p->Py) {
        auto kern = columns_lp_kernel<LGN, true>;
        if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(kern, dim3(grid), dim3(block), (size_t)(smem), st, la);
    } else {
        auto kern = columns_lp_kernel<LGN, false>;
        if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(kern, dim3(grid), dim3(block), (size_t)(smem), st, la);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
static int launch_columns_lp_any(const DemagPlan* p, const ColLPArgs& la, cudaStream_t st)
{
    switch (ilog2(p->Py)) {
        case 8: return launch_columns_lp<8>(p, la, st);
        case 9: return launch_columns_lp<9>(p, la, st);
        case 10: return launch_columns_lp<10>(p, la, st);
        case 11: return launch_columns_lp<11>(p, la, st);
        case 12: return launch_columns_lp<12>(p, la, st);
        default: return MMC_E_UNSUPPORTED;
    }
}

template <int LGN>
static int launch_columns8(const DemagPlan* p, const ColFastArgs& ca, cudaStream_t st)
{
    using S = fftr8::Shape<LGN>;
    const size_t smem = (size_t)S::SMEM * sizeof(float2);
    const dim3 grid(p->Pz, p->Cx), block(S::T);
    if (2 * p->g.ny == p->Py) {
        auto kern = columns8_kernel<LGN, true>;
        if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(kern, dim3(grid), dim3(block), (size_t)(smem), st, ca);
    } else {
        auto kern = columns8_kernel<LGN, false>;
        if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(kern, dim3(grid), dim3(block), (size_t)(smem), st, ca);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

static int launch_columns_fast_any(const DemagPlan* p, const ColFastArgs& ca, cudaStream_t st)
{
    if (p->cols8) {
        switch (ilog2(p->Py)) {
            case 10: return launch_columns8<10>(p, ca, st);
            case 11: return launch_columns8<11>(p, ca, st);
            case 12: return launch_columns8<12>(p, ca, st);
            default: return MMC_E_UNSUPPORTED;
        }
    }
    switch (ilog2(p->Py)) {
        case 8: return launch_columns_fast<8>(p, ca, st);
        case 9: return launch_columns_fast<9>(p, ca, st);
        case 10: return launch_columns_fast<10>(p, ca, st);
        case 11: return launch_columns_fast<11>(p, ca, st);
        case 12: return launch_columns_fast<12>(p, ca, st);
        default: return MMC_E_UNSUPPORTED;
    }
}

// ------------------------------------------------------------------------------------------------ host side
template <int PZ>
static int launch_rows(const DemagPlan* p, const RowArgs& ra, bool inverse, cudaStream_t st)
{
    const dim3 grid((p->g.ny + p->RJ - 1) / p->RJ, 3);
    if (inverse) {
        if (p->smemA > 48 * 1024 && cudaFuncSetAttribute(rows_inv_kernel<PZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smemA) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(rows_inv_kernel<PZ>, dim3(grid), dim3(p->threadsA), p->smemA, st, ra);
    } else {
        if (p->smemA > 48 * 1024 && cudaFuncSetAttribute(rows_fwd_kernel<PZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smemA) != cudaSuccess) return MMC_E_CUDA;
        launch_pdl(rows_fwd_kernel<PZ>, dim3(grid), dim3(p->threadsA), p->smemA, st, ra);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
static int launch_rows_any(const DemagPlan* p, const RowArgs& ra, bool inverse, cudaStream_t st)
{
    switch (p->lgPz) {
        case 0: return launch_rows<1>(p, ra, inverse, st);
        case 1: return launch_rows<2>(p, ra, inverse, st);
        case 2: return launch_rows<4>(p, ra, inverse, st);
        case 3: return launch_rows<8>(p, ra, inverse, st);
        case 4: return launch_rows<16>(p, ra, inverse, st);
        case 5: return launch_rows<32>(p, ra, inverse, st);
        default: return MMC_E_UNSUPPORTED;
    }
}

int demag_create(DemagPlan** out, const Geometry& g, double dx, double dy, double dz, void* stream, std::string* err)
{
    cudaStream_t st = (cudaStream_t)stream;
    DemagPlan* p = new DemagPlan();
    *out = p;
    p->g = g;
    p->Px = padded_pow2(g.nx, 2); p->Py = padded_pow2(g.ny, 1); p->Pz = padded_pow2(g.nz, 1);
    p->Hx = p->Px / 2; p->Cx = p->Hx + 1;
    {
        // register-resident path: per-layer rows kernels, z-DFT outside them (fused into the columns kernel's load, and
        // the z_inverse pass).  Its z length is the SHORTEST that makes the cyclic convolution linear, Pz = 2 nz - 1
        // (7 planes instead of 8 for four layers, 5 instead of 8 for three): the z-DFT is a direct sum there, so any
        // length will do, and every plane saved is a whole set of column transforms saved.
        const int lgH = ilog2(p->Hx), lgPy = ilog2(p->Py);
        p->fastA = lgH >= 8 && lgH <= 11 && lgPy >= fftr::kMinLg && lgPy <= fftr::kMaxLg && g.nz <= kMaxFastLayers;
        // MMC_DEMAG_GENERIC=1 (tests): the any-length shared-memory kernels on meshes the register-resident ones would serve
        { const char* e = std::getenv("MMC_DEMAG_GENERIC"); if (e && e[0] == '1') p->fastA = false; }
        if (p->fastA && g.nz > 1) p->Pz = 2 * g.nz - 1;
    }
    p->lgPz = ilog2(p->Pz);
    p->px = fft::make_plan(ilog2(p->Hx)); p->py = fft::make_plan(ilog2(p->Py));
    if (p->lgPz > 5) { if (err) *err = "demag: more than 16 layers (padded z length > 32) is not built"; return MMC_E_UNSUPPORTED; }
    // kernels A/C: rows per CTA.  8 if that leaves room for two CTAs per SM, else 4 (32-byte store segments), less
    // only when even that does not fit the 227 KB of one SM.
    p->RS = fft::padded_len(p->Hx) + 1;
    auto bytesA = [&](int rj) { return (size_t)rj * g.nz * p->RS * sizeof(float2); };
    p->RJ = 8;
    while (p->RJ > 4 && bytesA(p->RJ) > 100 * 1024) p->RJ >>= 1;
    while (p->RJ > 1 && bytesA(p->RJ) > 200 * 1024) p->RJ >>= 1;
    while (p->RJ > 1 && p->RJ / 2 >= g.ny) p->RJ >>= 1;
    if (!p->fastA && bytesA(p->RJ) > 220 * 1024) { if (err) *err = "demag: nz * padded nx too large for the fused row kernels"; return MMC_E_UNSUPPORTED; }
    p->smemA = bytesA(p->RJ);
    p->threadsA = p->smemA > 100 * 1024 ? 512 : 256;
    p->smemB = (size_t)3 * fft::padded_len(p->Py) * sizeof(float2);
    if (p->smemB > 220 * 1024) { if (err) *err = "demag: padded ny > 8192 is not built"; return MMC_E_UNSUPPORTED; }
    { int t = (3 * p->Py / 16 + 31) / 32 * 32; p->threadsB = t < 32 ? 32 : (t > 256 ? 256 : t); }

    {
        const int lgPy = ilog2(p->Py);
        p->fastB = lgPy >= fftr::kMinLg && lgPy <= fftr::kMaxLg;
        { const char* e = std::getenv("MMC_DEMAG_GENERIC"); if (e && e[0] == '1') p->fastB = false; }
        if (p->fastB) {
            const size_t ntw = (size_t)15 * (p->Py / 16);
            CK(cudaMalloc(&p->twB1, ntw * sizeof(float2)));
            CK(cudaMalloc(&p->twB2, ntw * sizeof(float2)));
            fftr::twiddle_tables_kernel<<<blocks_for((long long)ntw), 256, 0, st>>>(p->twB1, p->twB2, lgPy);
        }
    }
    if (p->fastB && g.nz == 1) {
        // Measured (ms per iteration, cfg 2 / cfg 3 / cfg 5): one CTA for all three components 0.0225 / 0.0293 / 0.3727; pair and z
        // in separate CTAs 0.0209 / 0.0286 / 0.3738; every component in its own thread group of a 256-thread CTA, the pair meeting
        // in shared memory, 0.0219 / 0.0308 / 0.412 (CTA-wide barriers over twice the warps).  MMC_COLS_SPLIT=0/1 forces the choice.
        const int Tn = p->Py / 16, G = Tn >= 128 ? 1 : 128 / Tn;       // fftr::Shape<lgPy>::T, ::G
        const char* e = std::getenv("MMC_COLS_SPLIT");
        p->planar_split = e ? e[0] == '1' : (p->Cx + G - 1) / G < 2 * 148;
    }
    // several layers on the register-resident path: the layer-pair columns kernel when one CTA can hold a thread group per
    // layer (nz * Py/16 <= 512 threads); else the z-DFT path (planes T, z_inverse pass)
#ifndef MMC_DEMAG_LP
#define MMC_DEMAG_LP 0
#endif
    {
        const int Tn = p->Py / 16;
        // Measured on BASELINE config 4 (1024 x 1024 x 4): layer-pair 0.314 ms against 0.240 + 0.045 ms for the z-DFT columns kernel
        // + inverse z pass: the z-DFT path is the default, the layer-pair kernel is selected with MMC_LP=1
        const char* lp_env = std::getenv("MMC_LP");
        const bool lp_on = lp_env ? lp_env[0] == '1' : (MMC_DEMAG_LP != 0);
        p->lp = lp_on && p->fastA && g.nz > 1 && Tn * g.nz <= 512;
        if (p->lp) {
            const int gmax = std::max(1, std::min(Tn >= 128 ? 1 : 128 / Tn, 512 / (Tn * g.nz)));
            p->lpG = std::min(gmax, std::max(1, p->Cx / 296));          // short transforms share a CTA once the grid is two waves deep
            while (p->lpG > 1 && lp_smem_bytes_any(ilog2(p->Py), g.nz, p->lpG) > 227 * 1024) p->lpG >>= 1;
            if (lp_smem_bytes_any(ilog2(p->Py), g.nz, p->lpG) > 227 * 1024) p->lp = false;      // does not fit one SM: the z-DFT path
        }
    }
#ifndef MMC_DEMAG_COLS8
#define MMC_DEMAG_COLS8 0
#endif
    {
        // eight points per thread in the columns kernel of the z-DFT path (MMC_COLS8=0/1 forces the choice)
        const int lgPy = ilog2(p->Py);
        const char* e = std::getenv("MMC_COLS8");
        const bool on = e ? e[0] == '1' : (MMC_DEMAG_COLS8 != 0);
        p->cols8 = on && !p->lp && p->fastA && p->fastB && g.nz > 1 && lgPy >= fftr8::kMinLg && lgPy <= fftr8::kMaxLg && p->Cx <= 65535;
        if (p->cols8) {
            const int ntw = 7 * (p->Py / 8 + p->Py / 64 + p->Py / 512);
            CK(cudaMalloc(&p->tw8, (size_t)ntw * sizeof(float2)));
            fftr8::twiddle_tables8_kernel<<<blocks_for(ntw), 256, 0, st>>>(p->tw8, lgPy);
        }
    }
    const size_t nT = (size_t)3 * p->Pz * p->Cx * g.ny;
    if (!p->lp) CK(cudaMalloc(&p->T, nT * sizeof(float2)));
    if (p->fastA && g.nz > 1) CK(cudaMalloc(&p->U, (size_t)3 * g.nz * p->Cx * g.ny * sizeof(float2)));
    CK(cudaMalloc(&p->twx, (size_t)p->Px * sizeof(float2)));
    CK(cudaMalloc(&p->twy, (size_t)p->Py * sizeof(float2)));
    twiddle_kernel<<<blocks_for(p->Px), 256, 0, st>>>(p->twx, p->Px);
    twiddle_kernel<<<blocks_for(p->Py), 256, 0, st>>>(p->twy, p->Py);

    // tensor spectrum, fp64 set-up
    std::vector<double> oct[6];
    demag_tensor_octant(g.nx, g.ny, g.nz, dx, dy, dz, kNearRadius, oct);
    const size_t nO = (size_t)g.nx * g.ny * g.nz;
    static const int SX[6] = { 1, 1, 1, -1, -1, 1 }, SY[6] = { 1, 1, 1, -1, 1, -1 }, SZ[6] = { 1, 1, 1, 1, -1, -1 };
    if (p->lp) {
        // 2-D spectra of the tensor at every layer offset dz = 0 .. nz-1 (the octant table holds dz >= 0; the kernel applies the
        // parity in dz): place plane dz on the (Px, Py) grid, 2-D D2Z, real part (xx, yy, zz, xy) or imaginary part (xz, yz: odd
        // in exactly one in-plane coordinate), in the column transform's slot order, -mu0 / (2 Px Py) folded in
        const size_t r2 = (size_t)p->Px * p->Py, c2 = (size_t)p->Cx * p->Py, nP = (size_t)g.nx * g.ny;
        double *d_oct = nullptr, *d_full = nullptr; double2* d_spec = nullptr;
        CK(cudaMalloc(&d_oct, nO * sizeof(double)));
        CK(cudaMalloc(&d_full, r2 * sizeof(double)));
        CK(cudaMalloc(&d_spec, c2 * sizeof(double2)));
        int n2[2] = { p->Py, p->Px };
        cufftHandle pd;
        CF(cufftPlanMany(&pd, 2, n2, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 1));
        CF(cufftSetStream(pd, st));
        const double scale2 = -kMu0 / (2.0 * (double)p->Px * (double)p->Py);
        for (int q = 0; q < 6; ++q) {
            CK(cudaMalloc(&p->nh2[q], (size_t)g.nz * c2 * sizeof(float)));
            CK(cudaMemsetAsync(p->nh2[q], 0, (size_t)g.nz * c2 * sizeof(float), st));
            CK(cudaMemcpyAsync(d_oct, oct[q].data(), nO * sizeof(double), cudaMemcpyHostToDevice, st));
            for (int dzp = (q >= 4 ? 1 : 0); dzp < g.nz; ++dzp) {        // xz, yz vanish at dz = 0
                place_kernel<<<blocks_for((long long)r2), 256, 0, st>>>(g.nx, g.ny, 1, p->Px, p->Py, 1, d_oct + (size_t)dzp * nP, SX[q], SY[q], 1, d_full);
                CF(cufftExecD2Z(pd, d_full, (cufftDoubleComplex*)d_spec));
                permute_kernel<<<blocks_for((long long)c2), 256, 0, st>>>(d_spec, p->nh2[q] + (size_t)dzp * c2, p->Cx, p->Py, 1, p->py, scale2,
                                                                         ilog2(p->Py), q >= 4 ? 1 : 0);
            }
            CK(cudaStreamSynchronize(st));                   // oct[q] host buffer must outlive the copy
        }
        cufftDestroy(pd);
        cudaFree(d_oct); cudaFree(d_full); cudaFree(d_spec);
        CK(cudaGetLastError());
        return MMC_OK;
    }
    const size_t rsize = (size_t)p->Px * p->Py * p->Pz, csize = (size_t)p->Cx * p->Py * p->Pz;
    const int Kz = p->Pz / 2 + 1;
    double *d_oct = nullptr, *d_full = nullptr; double2* d_spec = nullptr;
    CK(cudaMalloc(&d_oct, nO * sizeof(double)));
    CK(cudaMalloc(&d_full, rsize * sizeof(double)));
    CK(cudaMalloc(&d_spec, csize * sizeof(double2)));
    int n3[3] = { p->Pz, p->Py, p->Px };
    int rank = 3; int* dims = n3;
    if (p->Pz == 1) { rank = 2; dims = n3 + 1; }
    if (p->Pz == 1 && p->Py == 1) { rank = 1; dims = n3 + 2; }
    cufftHandle pd;
    CF(cufftPlanMany(&pd, rank, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 1));
    CF(cufftSetStream(pd, st));
    const double scale = -kMu0 / (2.0 * (double)p->Px * (double)p->Py * (double)p->Pz);
    for (int q = 0; q < 6; ++q) {
        if (g.nz == 1 && q >= 4) continue;                   // N_xz = N_yz = 0 in a single layer
        const size_t nN = (size_t)Kz * p->Cx * p->Py;
        CK(cudaMalloc(&p->nhat[q], nN * sizeof(float)));
        CK(cudaMemcpyAsync(d_oct, oct[q].data(), nO * sizeof(double), cudaMemcpyHostToDevice, st));
        place_kernel<<<blocks_for((long long)rsize), 256, 0, st>>>(g.nx, g.ny, g.nz, p->Px, p->Py, p->Pz, d_oct, SX[q], SY[q], SZ[q], d_full);
        CF(cufftExecD2Z(pd, d_full, (cufftDoubleComplex*)d_spec));
        permute_kernel<<<blocks_for((long long)nN), 256, 0, st>>>(d_spec, p->nhat[q], p->Cx, p->Py, Kz, p->py, scale,
                                                                  p->cols8 ? -ilog2(p->Py) : p->fastB ? ilog2(p->Py) : 0);
        CK(cudaStreamSynchronize(st));                       // oct[q] host buffer must outlive the copy
    }
    cufftDestroy(pd);
    cudaFree(d_oct); cudaFree(d_full); cudaFree(d_spec);
    if (p->smemB > 48 * 1024) {
        CK(cudaFuncSetAttribute(columns_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smemB));
        CK(cudaFuncSetAttribute(columns_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smemB));
    }
    CK(cudaGetLastError());
    return MMC_OK;
}

void demag_destroy(DemagPlan* p)
{
    if (!p) return;
    cudaFree(p->T); cudaFree(p->U); cudaFree(p->twx); cudaFree(p->twy); cudaFree(p->twB1); cudaFree(p->twB2); cudaFree(p->tw8);
    for (int q = 0; q < 6; ++q) { cudaFree(p->nhat[q]); cudaFree(p->nh2[q]); }
    delete p;
}

void PhaseTimer::mark(int ph, void* stream)
{
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess || cudaEventRecord(e, (cudaStream_t)stream) != cudaSuccess) { failed = true; return; }   // mmc_sweep_timed reports it
    events.push_back((void*)e); phase.push_back(ph);
}

int demag_compute(DemagPlan* p, const float* const m[3], const float* Ms0_split, float Ms0_uniform, float* const bd[3],
                  void* stream, std::string* err, PhaseTimer* timer)
{
    cudaStream_t st = (cudaStream_t)stream;
    RowArgs ra{};
    ra.g = p->g; ra.Hx = p->Hx; ra.lgHx = ilog2(p->Hx); ra.Cx = p->Cx; ra.lgPx = ilog2(p->Px);
    ra.RJ = p->RJ; ra.lgRJ = ilog2(p->RJ); ra.RS = p->RS; ra.px = p->px; ra.twx = p->twx;
    for (int c = 0; c < 3; ++c) { ra.m[c] = m[c]; ra.bd[c] = bd[c]; }
    ra.Ms0 = Ms0_split; ra.Ms0_u = Ms0_uniform; ra.T = p->T;
    RowFastArgs rf{};
    rf.g = p->g; rf.Cx = p->Cx;
    if (p->fastA) {
        const int lgH = ilog2(p->Hx);
        for (int e = 0; e < 16; ++e) {                      // kconst(e) of fft_reg.cuh = freq_of_slot(thread 0, e)
            const double ang = -2.0 * M_PI * (double)fftr::freq_of_slot(lgH, 0, e) / (double)p->Px;
            rf.cu[e] = make_float2((float)std::cos(ang), (float)std::sin(ang));
        }
    }
    for (int c = 0; c < 3; ++c) { rf.m[c] = m[c]; rf.bd[c] = bd[c]; }
    rf.Ms0 = Ms0_split; rf.Ms0_u = Ms0_uniform; rf.T = p->U ? p->U : p->T;
    int rc = p->fastA ? launch_rows_fast_any(p, rf, false, st) : launch_rows_any(p, ra, false, st);
    if (rc) { if (err) *err = "rows_fwd_kernel launch failed"; return rc; }
    if (timer) timer->mark(PH_FFT_FWD, stream);
    ColArgs ca{};
    ca.ny = p->g.ny; ca.Cx = p->Cx; ca.Py = p->Py; ca.lgPy = ilog2(p->Py); ca.Pz = p->Pz; ca.BS = fft::padded_len(p->Py);
    ca.py = p->py; ca.twy = p->twy; ca.T = p->T;
    for (int q = 0; q < 6; ++q) ca.nhat[q] = p->nhat[q];
    if (p->lp) {
        ColLPArgs la{};
        la.ny = p->g.ny; la.Cx = p->Cx; la.tw1 = p->twB1; la.tw2 = p->twB2; la.U = p->U;
        for (int q = 0; q < 6; ++q) la.nh[q] = p->nh2[q];
        rc = launch_columns_lp_any(p, la, st);
        if (rc) { if (err) *err = "columns_lp_kernel launch failed"; return rc; }
        if (timer) timer->mark(PH_MULTIPLY, stream);
    } else if (p->fastB) {
        ColFastArgs fa{};
        fa.ny = p->g.ny; fa.Cx = p->Cx; fa.Pz = p->Pz; fa.nz = p->U ? p->g.nz : 0; fa.tw1 = p->twB1; fa.tw2 = p->twB2;
        fa.Tin = p->U ? p->U : p->T; fa.Tout = p->T;
        if (p->cols8) fa.tw1 = p->tw8;
        for (int q = 0; q < 6; ++q) fa.nhat[q] = p->nhat[q];
        rc = launch_columns_fast_any(p, fa, st);
        if (rc) { if (err) *err = "columns_fast_kernel launch failed"; return rc; }
        if (timer) timer->mark(PH_MULTIPLY, stream);
        if (p->U) {
            rc = launch_z_inverse(p, p->T, p->U, st);
            if (rc) { if (err) *err = "z_inverse_kernel launch failed"; return rc; }
            if (timer) timer->mark(PH_CROP, stream);
        }
    } else {
        const dim3 gridB(p->Cx, p->Pz);
        if (p->g.nz > 1) launch_pdl(columns_kernel<true>, dim3(gridB), dim3(p->threadsB), p->smemB, st, ca);
        else             launch_pdl(columns_kernel<false>, dim3(gridB), dim3(p->threadsB), p->smemB, st, ca);
        if (timer) timer->mark(PH_MULTIPLY, stream);
    }
    rc = p->fastA ? launch_rows_fast_any(p, rf, true, st) : launch_rows_any(p, ra, true, st);
    if (rc) { if (err) *err = "rows_inv_kernel launch failed"; return rc; }
    if (timer) timer->mark(PH_FFT_INV, stream);
    CK(cudaGetLastError());
    return MMC_OK;
}

}  // namespace mmc
