// demag.cu -- demagnetising field of Eq. (14): B_d = -mu0 N (*) M by zero-padded FFT convolution.
//   S0 pack + pad (M = Ms0 m from the colour-split state)      -> pack_kernel
//   S1 forward real-to-complex FFT of the three components     -> cuFFT (round-1 baseline)
//   S2 tensor multiply with the real-valued spectrum of N      -> multiply_kernel
//   S3 inverse FFT + crop to the N physical cells              -> cuFFT + crop_kernel (writes colour-split B_d)
// The tensor spectrum is built once at set-up in fp64 (host Newell/moment table -> device placement -> D2Z) and kept
// in fp32 with the factor -mu0/(Px Py Pz) folded in.
#include <cuda_runtime.h>
#include <cufft.h>

#include "mmc_internal.h"

namespace mmc {

struct DemagPlan {
    Geometry g;
    int Px, Py, Pz, Cx;              // padded real dims, complex x length Px/2+1
    size_t rsize, csize;             // elements per component
    float* rbuf = nullptr;           // 3 * rsize, zero outside the physical block (never written there)
    float* obuf = nullptr;           // 3 * rsize, inverse-transform output
    float2* cbuf = nullptr;          // 3 * csize
    float* khat[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
    cufftHandle fwd = 0, inv = 0;
    bool have_fwd = false, have_inv = false;
};

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { if (err) *err = std::string(#x) + ": " + cudaGetErrorString(e_); return MMC_E_CUDA; } } while (0)
#define CF(x) do { cufftResult r_ = (x); if (r_ != CUFFT_SUCCESS) { if (err) *err = std::string(#x) + ": cufft error " + std::to_string((int)r_); return MMC_E_CUDA; } } while (0)

// place the octant table on the padded periodic grid: offset o_d (|o_d| < N_d) at index o_d mod P_d, index N_d zero;
// diagonal components even, N_ab odd in coordinates a and b.
__global__ void place_kernel(int nx, int ny, int nz, int Px, int Py, int Pz, const double* __restrict__ oct, int sx, int sy, int sz,
                             double* __restrict__ full)
{
    const long long n = (long long)Px * Py * Pz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(t % Px); const long long r = t / Px; const int y = (int)(r % Py), z = (int)(r / Py);
        int ox = x < nx ? x : x - Px, oy = y < ny ? y : y - Py, oz = z < nz ? z : z - Pz;
        double v = 0.0;
        const bool hole = (Px > 1 && x == nx) || (Py > 1 && y == ny) || (Pz > 1 && z == nz);
        if (!hole) {
            double s = 1.0;
            if (ox < 0) { ox = -ox; s *= sx; }
            if (oy < 0) { oy = -oy; s *= sy; }
            if (oz < 0) { oz = -oz; s *= sz; }
            v = s * oct[((long long)oz * ny + oy) * nx + ox];
        }
        full[t] = v;
    }
}
__global__ void real_part_kernel(const double2* __restrict__ z, float* __restrict__ out, long long n, double scale)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        out[t] = (float)(scale * z[t].x);
}

static int blocks_for(long long n) { long long b = (n + 255) / 256; return (int)(b > 148 * 32 ? 148 * 32 : (b < 1 ? 1 : b)); }

int demag_create(DemagPlan** out, const Geometry& g, double dx, double dy, double dz, void* stream, std::string* err)
{
    cudaStream_t st = (cudaStream_t)stream;
    DemagPlan* p = new DemagPlan();
    p->g = g;
    p->Px = g.nx > 1 ? 2 * g.nx : 1; p->Py = g.ny > 1 ? 2 * g.ny : 1; p->Pz = g.nz > 1 ? 2 * g.nz : 1;
    p->Cx = p->Px / 2 + 1;
    p->rsize = (size_t)p->Px * p->Py * p->Pz;
    p->csize = (size_t)p->Cx * p->Py * p->Pz;
    *out = p;
    CK(cudaMalloc(&p->rbuf, 3 * p->rsize * sizeof(float)));
    CK(cudaMalloc(&p->obuf, 3 * p->rsize * sizeof(float)));
    CK(cudaMalloc(&p->cbuf, 3 * p->csize * sizeof(float2)));
    CK(cudaMemsetAsync(p->rbuf, 0, 3 * p->rsize * sizeof(float), st));
    int n3[3] = { p->Pz, p->Py, p->Px };
    int rank = 3; int* dims = n3;
    if (p->Pz == 1) { rank = 2; dims = n3 + 1; }
    if (p->Pz == 1 && p->Py == 1) { rank = 1; dims = n3 + 2; }
    CF(cufftPlanMany(&p->fwd, rank, dims, nullptr, 1, (int)p->rsize, nullptr, 1, (int)p->csize, CUFFT_R2C, 3)); p->have_fwd = true;
    CF(cufftPlanMany(&p->inv, rank, dims, nullptr, 1, (int)p->csize, nullptr, 1, (int)p->rsize, CUFFT_C2R, 3)); p->have_inv = true;
    CF(cufftSetStream(p->fwd, st));
    CF(cufftSetStream(p->inv, st));

    // tensor spectrum, fp64 set-up
    std::vector<double> oct[6];
    demag_tensor_octant(g.nx, g.ny, g.nz, dx, dy, dz, kNearRadius, oct);
    const size_t nO = (size_t)g.nx * g.ny * g.nz;
    double *d_oct = nullptr, *d_full = nullptr; double2* d_spec = nullptr;
    CK(cudaMalloc(&d_oct, nO * sizeof(double)));
    CK(cudaMalloc(&d_full, p->rsize * sizeof(double)));
    CK(cudaMalloc(&d_spec, p->csize * sizeof(double2)));
    cufftHandle pd;
    CF(cufftPlanMany(&pd, rank, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 1));
    CF(cufftSetStream(pd, st));
    static const int SX[6] = { 1, 1, 1, -1, -1, 1 }, SY[6] = { 1, 1, 1, -1, 1, -1 }, SZ[6] = { 1, 1, 1, 1, -1, -1 };
    const double scale = -kMu0 / (double)p->rsize;
    for (int q = 0; q < 6; ++q) {
        if (g.nz == 1 && q >= 4) continue;                   // N_xz = N_yz = 0 in a single layer
        CK(cudaMalloc(&p->khat[q], p->csize * sizeof(float)));
        CK(cudaMemcpyAsync(d_oct, oct[q].data(), nO * sizeof(double), cudaMemcpyHostToDevice, st));
        place_kernel<<<blocks_for((long long)p->rsize), 256, 0, st>>>(g.nx, g.ny, g.nz, p->Px, p->Py, p->Pz, d_oct, SX[q], SY[q], SZ[q], d_full);
        CF(cufftExecD2Z(pd, d_full, (cufftDoubleComplex*)d_spec));
        real_part_kernel<<<blocks_for((long long)p->csize), 256, 0, st>>>(d_spec, p->khat[q], (long long)p->csize, scale);
        CK(cudaStreamSynchronize(st));                       // oct[q] host buffer must outlive the copy
    }
    cufftDestroy(pd);
    cudaFree(d_oct); cudaFree(d_full); cudaFree(d_spec);
    CK(cudaGetLastError());
    return MMC_OK;
}

void demag_destroy(DemagPlan* p)
{
    if (!p) return;
    if (p->have_fwd) cufftDestroy(p->fwd);
    if (p->have_inv) cufftDestroy(p->inv);
    cudaFree(p->rbuf); cudaFree(p->obuf); cudaFree(p->cbuf);
    for (int q = 0; q < 6; ++q) cudaFree(p->khat[q]);
    delete p;
}

// S0: one thread per natural pair (i = 2p, 2p+1): one coalesced read from each colour array, one float2 store.
__global__ void __launch_bounds__(256) pack_kernel(Geometry g, int Px, int Py, size_t rsize, const float* __restrict__ mx, const float* __restrict__ my,
                            const float* __restrict__ mz, const float* __restrict__ Ms0, float Ms0_u, float* __restrict__ rbuf)
{
    const int hp = (g.nx + 1) >> 1;
    const long long n = (long long)hp * g.ny * g.nz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int p = (int)(t % hp); const long long row = t / hp;
        const int j = (int)(row % g.ny), k = (int)(row / g.ny);
        const int par = (j + k) & 1;
        const long long se = (long long)par * g.H + row * g.hx + p;          // cell i = 2p
        const long long so = (long long)(1 - par) * g.H + row * g.hx + p;    // cell i = 2p+1
        const float we = Ms0 ? Ms0[se] : Ms0_u;
        const bool has_odd = 2 * p + 1 < g.nx;
        const float wo = has_odd ? (Ms0 ? Ms0[so] : Ms0_u) : 0.f;
        const long long dst = ((long long)k * Py + j) * Px + 2 * p;
        const float* src[3] = { mx, my, mz };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float ve = we * src[c][se];
            const float vo = has_odd ? wo * src[c][so] : 0.f;
            float* d = rbuf + c * rsize + dst;
            if (Px > 1) *reinterpret_cast<float2*>(d) = make_float2(ve, vo);   // Px = 2 nx is even and dst is even
            else d[0] = ve;
        }
    }
}

// S2: B^ = K^ M^ with K^ = -mu0/(P) N^ real and symmetric.
template <bool THREE_D>
__global__ void __launch_bounds__(256) multiply_kernel(size_t csize, float2* __restrict__ c, const float* __restrict__ kxx, const float* __restrict__ kyy,
                                const float* __restrict__ kzz, const float* __restrict__ kxy, const float* __restrict__ kxz,
                                const float* __restrict__ kyz)
{
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < csize; t += (size_t)gridDim.x * blockDim.x) {
        const float2 a = c[t], b = c[csize + t], d = c[2 * csize + t];
        const float xx = kxx[t], yy = kyy[t], zz = kzz[t], xy = kxy[t];
        float2 ox, oy, oz;
        ox.x = xx * a.x + xy * b.x; ox.y = xx * a.y + xy * b.y;
        oy.x = xy * a.x + yy * b.x; oy.y = xy * a.y + yy * b.y;
        oz.x = zz * d.x;            oz.y = zz * d.y;
        if (THREE_D) {
            const float xz = kxz[t], yz = kyz[t];
            ox.x += xz * d.x; ox.y += xz * d.y;
            oy.x += yz * d.x; oy.y += yz * d.y;
            oz.x += xz * a.x + yz * b.x; oz.y += xz * a.y + yz * b.y;
        }
        c[t] = ox; c[csize + t] = oy; c[2 * csize + t] = oz;
    }
}

// S3 (crop): natural pair -> the two colour arrays of B_d.
__global__ void __launch_bounds__(256) crop_kernel(Geometry g, int Px, int Py, size_t rsize, const float* __restrict__ rbuf, float* __restrict__ bx,
                            float* __restrict__ by, float* __restrict__ bz)
{
    const int hp = (g.nx + 1) >> 1;
    const long long n = (long long)hp * g.ny * g.nz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const int p = (int)(t % hp); const long long row = t / hp;
        const int j = (int)(row % g.ny), k = (int)(row / g.ny);
        const int par = (j + k) & 1;
        const long long se = (long long)par * g.H + row * g.hx + p;
        const long long so = (long long)(1 - par) * g.H + row * g.hx + p;
        const bool has_odd = 2 * p + 1 < g.nx;
        const long long srcidx = ((long long)k * Py + j) * Px + 2 * p;
        float* dst[3] = { bx, by, bz };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* s = rbuf + c * rsize + srcidx;
            float ve, vo = 0.f;
            if (Px > 1) { const float2 v = *reinterpret_cast<const float2*>(s); ve = v.x; vo = v.y; }
            else ve = s[0];
            dst[c][se] = ve;
            if (has_odd) dst[c][so] = vo;
        }
    }
}

void PhaseTimer::mark(int ph, void* stream)
{
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, (cudaStream_t)stream);
    events.push_back((void*)e); phase.push_back(ph);
}

int demag_compute(DemagPlan* p, const float* const m[3], const float* Ms0_split, float Ms0_uniform, float* const bd[3],
                  void* stream, std::string* err, PhaseTimer* timer)
{
    cudaStream_t st = (cudaStream_t)stream;
    const Geometry& g = p->g;
    const long long pairs = (long long)((g.nx + 1) >> 1) * g.ny * g.nz;
    pack_kernel<<<blocks_for(pairs), 256, 0, st>>>(g, p->Px, p->Py, p->rsize, m[0], m[1], m[2], Ms0_split, Ms0_uniform, p->rbuf);
    if (timer) timer->mark(PH_PACK, stream);
    CF(cufftExecR2C(p->fwd, p->rbuf, (cufftComplex*)p->cbuf));
    if (timer) timer->mark(PH_FFT_FWD, stream);
    if (g.nz > 1)
        multiply_kernel<true><<<blocks_for((long long)p->csize), 256, 0, st>>>(p->csize, p->cbuf, p->khat[0], p->khat[1], p->khat[2], p->khat[3], p->khat[4], p->khat[5]);
    else
        multiply_kernel<false><<<blocks_for((long long)p->csize), 256, 0, st>>>(p->csize, p->cbuf, p->khat[0], p->khat[1], p->khat[2], p->khat[3], nullptr, nullptr);
    if (timer) timer->mark(PH_MULTIPLY, stream);
    CF(cufftExecC2R(p->inv, (cufftComplex*)p->cbuf, p->obuf));
    if (timer) timer->mark(PH_FFT_INV, stream);
    crop_kernel<<<blocks_for(pairs), 256, 0, st>>>(g, p->Px, p->Py, p->rsize, p->obuf, bd[0], bd[1], bd[2]);
    if (timer) timer->mark(PH_CROP, stream);
    CK(cudaGetLastError());
    return MMC_OK;
}

}  // namespace mmc
