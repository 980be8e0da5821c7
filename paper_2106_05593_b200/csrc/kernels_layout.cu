// kernels_layout.cu -- natural <-> colour-split layout conversion, the zero-length check of mmc_set_m, and the
// read-out reduction (means and energies with pair terms counted once).
#include <cuda_runtime.h>

#include <algorithm>

#include "mmc_internal.h"

namespace mmc {

__host__ __device__ inline long long split_index(const Geometry& g, int i, int j, int k)
{
    const int col = (i + j + k) & 1;
    return (long long)col * g.H + ((long long)k * g.ny + j) * g.hx + (i >> 1);
}

__global__ void to_split_kernel(Geometry g, const float* __restrict__ nat, float* __restrict__ split)
{
    const long long N = (long long)g.nx * g.ny * g.nz;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(c % g.nx); const long long r = c / g.nx;
        const int j = (int)(r % g.ny), k = (int)(r / g.ny);
        split[split_index(g, i, j, k)] = nat[c];
    }
}
__global__ void from_split_kernel(Geometry g, const float* __restrict__ split, float* __restrict__ nat)
{
    const long long N = (long long)g.nx * g.ny * g.nz;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(c % g.nx); const long long r = c / g.nx;
        const int j = (int)(r % g.ny), k = (int)(r / g.ny);
        nat[c] = split[split_index(g, i, j, k)];
    }
}
static int grid_for(long long n) { long long b = (n + 255) / 256; return (int)(b > 148 * 16 ? 148 * 16 : (b < 1 ? 1 : b)); }

int launch_to_split(const Geometry& g, const float* nat, float* split, void* stream)
{
    to_split_kernel<<<grid_for((long long)g.nx * g.ny * g.nz), 256, 0, (cudaStream_t)stream>>>(g, nat, split);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
int launch_from_split(const Geometry& g, const float* split, float* nat, void* stream)
{
    from_split_kernel<<<grid_for((long long)g.nx * g.ny * g.nz), 256, 0, (cudaStream_t)stream>>>(g, split, nat);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// State check of mmc_set_m over the storage slots.  Non-empty cells: flag bit 0 when |m| = 0 or not finite (G13: rotation
// undefined, a multiplicative length move cannot leave 0), bit 1 when |m| >= 2 (m = M/Ms0; the fixed-point
// running sums of the pass are exact for |m| < 2).  Empty cells and padding slots: set to 0, whatever the caller passed
// (NaN markers included), so that the 0/1 bond weights and Ms0 = 0 factors that multiply them can never produce a NaN.
__global__ void check_state_kernel(Geometry g, float* mx, float* my, float* mz, const uint8_t* mask, int* flag)
{
    const long long n = 2 * g.H;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        if (!(mask[s] & 0x40u)) { mx[s] = 0.f; my[s] = 0.f; mz[s] = 0.f; continue; }
        const float l2 = mx[s] * mx[s] + my[s] * my[s] + mz[s] * mz[s];
        if (!(l2 > 0.f) || !isfinite(l2)) atomicOr(flag, 1);
        else if (!(l2 < 4.f)) atomicOr(flag, 2);
    }
}
int launch_check_state(const Geometry& g, float* const m[3], const uint8_t* mask, int* flag, void* stream)
{
    check_state_kernel<<<grid_for(2 * g.H), 256, 0, (cudaStream_t)stream>>>(g, m[0], m[1], m[2], mask, flag);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// ------------------------------------------------------------------------------------------------ read-out
// One thread per storage slot.  Quantities per active cell (all fp64 accumulation from fp32 state):
//   sums: mx, my, mz, |m|
//   E_ex   = 1/2 sum_{bonded nb} (A0 V/h_d^2)|m - m_nb|^2        (each bond seen from both ends)
//   E_an   = V K1(T) - (V K1 me)(m.e)^2 ; E_zee = -V Ms0 m.B_ext ; E_dmi = -D0 V m.G ;
//   E_demag = -(V Ms0/2) m.B_d ; E_long = kB T [c4 (l2 - mu2)^2 + c0adj]
#ifndef MMC_OBS_MINB
#define MMC_OBS_MINB 5
#endif
constexpr int kObsThreads = 128;     // 128-thread CTAs: five of them fit one SM at 96 registers (two 256-thread CTAs would leave a fifth of the file unused)
template <bool PERCELL, bool DMI>
__global__ void __launch_bounds__(kObsThreads, MMC_OBS_MINB) observables_kernel(SweepArgs a, ObsParams op, double* scratch, ReadOut* __restrict__ out)
{
    const Geometry g = a.g;
    const unsigned hx = (unsigned)g.hx, H = (unsigned)g.H, n = 2u * H;    // mmc_create: 2 H < 2^31
    const int hxr = (g.nx + 1) >> 1;
    double acc[11];
#pragma unroll
    for (int t = 0; t < 11; ++t) acc[t] = 0.0;
    // one thread per storage slot, 32-bit index arithmetic, neighbours by their offsets in the other colour's plane (as in the
    // pass); the exchange energy counts every bond once, from its -x / -y / -z end (bits 0, 2, 4 of the mask byte).
    // The kernel waits on memory, not on arithmetic (ncu: 14 of 19 warp cycles per instruction on long_scoreboard at 24 warps
    // per SM), so the loads of a slot are issued in two batches instead of where they are used: everything whose address
    // follows from the slot index alone (state, class word, B_d, the neighbours -- unconditionally, at the cell's own
    // address when the bond is absent), then the class-table entries that need the class word; the NEXT slot's mask byte
    // is requested one iteration ahead.
    const unsigned stride = gridDim.x * blockDim.x;
    unsigned s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned mb = s < n ? a.mask[s] : 0u;
    const bool has_bd = a.bd[0] != nullptr;
    for (; s < n; s += stride) {
        const unsigned mb_now = mb;
        mb = (s + stride < n) ? a.mask[s + stride] : 0u;
        if (!(mb_now & 0x40u)) continue;
        const unsigned col = s >= H ? 1u : 0u, w = s - col * H;
        const unsigned row = w / hx; const int q = (int)(w - row * hx);
        const int k = (int)(row / (unsigned)g.ny), j = (int)(row - (unsigned)k * g.ny);
        const int sp = ((j + k) & 1) ^ (int)col;
        const unsigned oth = (1u - col) * H + row * hx + q;           // same compact index in the other colour's plane
        // offsets of the six neighbours relative to `oth` (only used when the bond bit is set, i.e. the neighbour exists)
        int off[6];
        off[0] = sp ? ((q + 1 < hxr) ? 1 : -q) : 0;                                       // +x
        off[1] = sp ? 0 : ((q > 0) ? -1 : hxr - 1);                                       // -x
        off[2] = (j + 1 < g.ny) ? (int)hx : -(g.ny - 1) * (int)hx;                        // +y
        off[3] = (j > 0) ? -(int)hx : (g.ny - 1) * (int)hx;                               // -y
        const int lay = g.ny * (int)hx;
        off[4] = (k + 1 < g.nz) ? lay : -(g.nz - 1) * lay;                                // +z
        off[5] = (k > 0) ? -lay : (g.nz - 1) * lay;                                       // -z
        // ---- batch 1
        const float mf[3] = { a.m[0][s], a.m[1][s], a.m[2][s] };
        const unsigned cls = PERCELL ? (a.cw[s] >> 7) : 0u;
        float bdv[3] = { 0.f, 0.f, 0.f };
        if (has_bd) { bdv[0] = a.bd[0][s]; bdv[1] = a.bd[1][s]; bdv[2] = a.bd[2][s]; }
        float nb6[6][3];
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            const bool need = (d & 1) == 0 || (DMI && d < 4);        // + directions for the exchange, E/W/N/S for the DMI vector
            if (!need) continue;
            const unsigned t = ((mb_now >> d) & 1u) ? oth + (unsigned)off[d] : s;
            nb6[d][0] = a.m[0][t]; nb6[d][1] = a.m[1][t]; nb6[d][2] = a.m[2][t];
        }
        // ---- batch 2: three 16-byte loads per table (ClassSlot order)
        float4 t0 = make_float4(0.f, 0.f, 0.f, 0.f), t1 = t0, t2 = t0, u0 = t0, u1 = t0, u2 = t0;
        const bool cubic_tab = PERCELL && a.table_cubic != nullptr;
        if (PERCELL) {
            const float4* t = a.table + (size_t)(kClassFloats / 4) * cls;
            t0 = __ldg(t); t1 = __ldg(t + 1); t2 = __ldg(t + 2);
            if (cubic_tab) { const float4* u = a.table_cubic + (size_t)(kClassFloats / 4) * cls; u0 = __ldg(u); u1 = __ldg(u + 1); u2 = __ldg(u + 2); }
        }
        // fp32 per-cell terms (differences, dot products: a few 1e-7 relative), fp64 where a bracket cancels (l2 - mu2, the
        // anisotropy constant against its (m.e)^2 term) and for every accumulation
        const double m[3] = { mf[0], mf[1], mf[2] };
        const double l2 = m[0] * m[0] + m[1] * m[1] + m[2] * m[2];
        acc[0] += m[0]; acc[1] += m[1]; acc[2] += m[2]; acc[3] += (double)sqrtf((float)l2); acc[10] += 1.0;
        float nbv[4][3];
        double eex = 0.0;
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            const bool need = (d & 1) == 0 || (DMI && d < 4);
            const bool bond = need && ((mb_now >> d) & 1u);
            float v0 = 0.f, v1 = 0.f, v2 = 0.f;
            if (need) { v0 = bond ? nb6[d][0] : 0.f; v1 = bond ? nb6[d][1] : 0.f; v2 = bond ? nb6[d][2] : 0.f; }
            if ((d & 1) == 0) {
                const float e0 = mf[0] - v0, e1 = mf[1] - v1, e2 = mf[2] - v2;
                const double e = op.aex[d >> 1] * (double)fmaf(e0, e0, fmaf(e1, e1, e2 * e2));
                eex += bond ? e : 0.0;
            }
            if (d < 4) { nbv[d][0] = v0; nbv[d][1] = v1; nbv[d][2] = v2; }
        }
        acc[4] += eex;
        float invT, bKq, bzee, c4, ax, ay, az, K1T, c0a; double mu2;
        if (PERCELL) {
            invT = t0.x; c4 = t0.y; mu2 = __hiloint2double(__float_as_int(t0.w), __float_as_int(t0.z));
            bKq = t1.x; bzee = t1.y; ax = t1.w; ay = t2.x; az = t2.y; K1T = t2.z; c0a = t2.w;
        } else {
            invT = 1.f / op.T_u; bKq = a.coef.bKq; bzee = a.coef.bzee; c4 = a.coef.c4;
            ax = a.coef.ax; ay = a.coef.ay; az = a.coef.az; mu2 = a.coef.mu2; K1T = op.K1T_u; c0a = op.c0_u;
        }
        const double kT = op.kB / (double)invT;
        const double me_ = m[0] * ax + m[1] * ay + m[2] * az;
        acc[5] += kT * ((double)K1T - (double)bKq * me_ * me_);
        {   // cubic anisotropy, Eq. (12): direction cosines with respect to the class's cubic axes
            float cb[9]; float bK1c, bK2c, bK2u = 0.f;
            if (PERCELL) {
                if (cubic_tab) {                                     // CS_BK1C, CS_BK2C, CS_CUB .. CS_CUB + 8, CS_BK2U
                    bK1c = u0.x; bK2c = u0.y; cb[0] = u0.z; cb[1] = u0.w; cb[2] = u1.x; cb[3] = u1.y; cb[4] = u1.z; cb[5] = u1.w;
                    cb[6] = u2.x; cb[7] = u2.y; cb[8] = u2.z; bK2u = u2.w;
                } else {
#pragma unroll
                    for (int t = 0; t < 9; ++t) cb[t] = a.coef.cub[t];
                    bK1c = 0.f; bK2c = 0.f;
                }
            } else {
#pragma unroll
                for (int t = 0; t < 9; ++t) cb[t] = a.coef.cub[t];
                bK1c = a.coef.bK1c; bK2c = a.coef.bK2c; bK2u = a.coef.bK2u;
            }
            if (bK2u != 0.f) { const double gq = mu2 - me_ * me_; acc[5] += kT * (double)bK2u * gq * gq; }      // V K2(T) [1 - (m.e)^2/me^2]^2
            if (bK1c != 0.f || bK2c != 0.f) {
                const double il = 1.0 / sqrt(l2);
                const double al = (m[0] * cb[0] + m[1] * cb[1] + m[2] * cb[2]) * il, be = (m[0] * cb[3] + m[1] * cb[4] + m[2] * cb[5]) * il,
                             ga = (m[0] * cb[6] + m[1] * cb[7] + m[2] * cb[8]) * il;
                const double A = al * al, B = be * be, G = ga * ga;
                acc[5] += kT * ((double)bK1c * (A * B + A * G + B * G) + (double)bK2c * A * B * G);
            }
        }
        acc[6] += -kT * (double)(bzee * fmaf(mf[0], a.coef.Bx, fmaf(mf[1], a.coef.By, mf[2] * a.coef.Bz)));
        if (DMI) {
            const float ix = (float)op.inv_d[0], iy = (float)op.inv_d[1];
            const float G0 = 0.5f * (-(nbv[0][2] - nbv[1][2]) * ix);
            const float G1 = 0.5f * (-(nbv[2][2] - nbv[3][2]) * iy);
            const float G2 = 0.5f * ((nbv[0][0] - nbv[1][0]) * ix + (nbv[2][1] - nbv[3][1]) * iy);
            acc[7] += -op.D0V * (double)fmaf(mf[0], G0, fmaf(mf[1], G1, mf[2] * G2));
        }
        if (has_bd) acc[8] += -0.5 * kT * (double)(bzee * fmaf(mf[0], bdv[0], fmaf(mf[1], bdv[1], mf[2] * bdv[2])));
        const double dv = l2 - mu2;
        acc[9] += kT * ((double)c4 * dv * dv + (double)c0a);
    }
    __shared__ double sh[kObsThreads / 32][11];
    __shared__ bool s_last;
#pragma unroll
    for (int t = 0; t < 11; ++t) {
        double v = acc[t];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5][t] = v;
    }
    __syncthreads();
    if (threadIdx.x < 11) {
        double v = 0.0;
        for (int w = 0; w < kObsThreads / 32; ++w) v += sh[w][threadIdx.x];
        scratch[1 + 11ll * blockIdx.x + threadIdx.x] = v;
        __threadfence();                                             // the partial is visible before the ticket is drawn
    }
    __syncthreads();
    // the CTA that draws the last ticket finishes the read-out (no second launch): it sums the CTAs' partials in a fixed order
    // (deterministic), gathers the control block and the running sums beside them -- one device-to-host copy brings it all --
    // and leaves the ticket at zero for the next call.  The ticket is scratch[0], the partials follow.
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    if (threadIdx.x == 0) s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int t = warp; t < 11; t += kObsThreads / 32) {              // lane l takes CTAs l, l + 32, ... in order, then a fixed shuffle tree
        double v = 0.0;
        for (unsigned b = lane; b < gridDim.x; b += 32) v += __ldcg(scratch + 1 + 11ll * b + t);
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) {
            if (t < 4) out->obs.sum[t] = v;
            else if (t < 10) out->obs.E[t - 4] = v;
            else out->obs.n_active = (unsigned long long)(v + 0.5);
        }
    }
    if (threadIdx.x == 0) {
        out->ctl = *a.ctl;
#pragma unroll
        for (int q = 0; q < 4; ++q) out->run_sums[q] = a.run_sums ? a.run_sums[q] : 0ull;
        *ticket = 0u;
    }
}

// Histograms of the current state over the non-empty cells.  kind 0: x = |m|; kind 1: x = polar angle
// (radians) between m and the direction (dx, dy, dz).  Everything in fp64 from the fp32 state, bin = floor((x - lo) * scale),
// scale = nbins / (hi - lo); out-of-range values go to under/over.  Shared-memory counters per CTA, 64-bit global atomics:
// exact integers, order-independent.
__global__ void __launch_bounds__(256) histogram_kernel(Geometry g, const float* __restrict__ mx, const float* __restrict__ my,
                                                        const float* __restrict__ mz, const uint8_t* __restrict__ mask, int kind,
                                                        double dx, double dy, double dz, int nbins, double lo, double scale,
                                                        unsigned long long* __restrict__ counts /* nbins + 2 */)
{
    extern __shared__ unsigned int h[];
    for (int b = threadIdx.x; b < nbins + 2; b += blockDim.x) h[b] = 0u;
    __syncthreads();
    const long long n = 2 * g.H;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
        if (!(mask[s] & 0x40u)) continue;
        const double a = mx[s], b = my[s], c = mz[s];
        const double len = sqrt(a * a + b * b + c * c);
        double x = len;
        if (kind == 1) {
            double cs = (a * dx + b * dy + c * dz) / len;
            cs = cs > 1.0 ? 1.0 : (cs < -1.0 ? -1.0 : cs);
            x = acos(cs);
        }
        const double t = (x - lo) * scale;
        int bin;
        if (!(t >= 0.0)) bin = nbins;                    // under (also NaN)
        else if (t >= (double)nbins) bin = nbins + 1;    // over
        else bin = (int)t;
        atomicAdd(&h[bin], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins + 2; b += blockDim.x)
        if (h[b]) atomicAdd(&counts[b], (unsigned long long)h[b]);
}

int launch_histogram(const Geometry& g, const float* const m[3], const uint8_t* mask, int kind, const double dir[3], int nbins,
                     double lo, double hi, unsigned long long* dev_counts, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemsetAsync(dev_counts, 0, (size_t)(nbins + 2) * sizeof(unsigned long long), st) != cudaSuccess) return MMC_E_CUDA;
    const long long n = 2 * g.H;
    const int blocks = (int)std::min<long long>((n + 255) / 256, 148 * 8);
    histogram_kernel<<<blocks, 256, (size_t)(nbins + 2) * sizeof(unsigned int), st>>>(g, m[0], m[1], m[2], mask, kind, dir[0], dir[1], dir[2],
                                                                                    nbins, lo, (double)nbins / (hi - lo), dev_counts);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// scratch: the ticket word (zero at the first launch; every launch leaves it zero), then 11 doubles per CTA
int launch_observables(const SweepArgs& a, bool percell, const ObsParams& op, ReadOut* dev_out, double* scratch,
                            int scratch_blocks, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const bool dmi = op.D0V != 0.0;
    // scratch_blocks CTAs at most (the scratch holds their partials); small meshes get one slot per thread
    const long long slots = 2 * a.g.H;
    const int blocks = (int)std::max<long long>(1, std::min<long long>(scratch_blocks, (slots + kObsThreads - 1) / kObsThreads));
    if (percell) { if (dmi) observables_kernel<true, true><<<blocks, kObsThreads, 0, st>>>(a, op, scratch, dev_out);
                   else     observables_kernel<true, false><<<blocks, kObsThreads, 0, st>>>(a, op, scratch, dev_out); }
    else         { if (dmi) observables_kernel<false, true><<<blocks, kObsThreads, 0, st>>>(a, op, scratch, dev_out);
                   else     observables_kernel<false, false><<<blocks, kObsThreads, 0, st>>>(a, op, scratch, dev_out); }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

}  // namespace mmc
