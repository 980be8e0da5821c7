// fft_smem.cuh -- in-place power-of-two complex FFTs in shared memory for the demag convolution (demag.cu).
//
// Forward transforms are decimation-in-frequency (natural order in, digit-reversed order out), inverse transforms are
// the exact stage-by-stage mirror (decimation-in-time, digit-reversed in, natural out).  The convolution multiplies
// in the digit-reversed order (the tensor spectrum is stored in that order), so no reordering pass is ever needed.
// A transform of length P = 2^lgP is a sequence of radix-16/8/4/2 stages; each stage keeps R points of one
// butterfly in registers.  Shared-memory index i is stored at pad(i) = i + (i >> 4): with 8-byte elements this makes
// every stage's access pattern (stride M = 1 ... P/R between the lanes' points) hit each bank pair exactly twice per
// warp, the minimum for 64-bit accesses.
#ifndef MMC_FFT_SMEM_CUH_
#define MMC_FFT_SMEM_CUH_

#include <cuda_runtime.h>

namespace mmc {
namespace fft {

struct Plan {               // stage radices of one transform length, as log2 (4, 3, 2, 1), in forward order
    int lgP;
    int nstages;
    int lgR[8];
};

__host__ __device__ inline int pad(int i) { return i + (i >> 4); }
__host__ __device__ inline int padded_len(int P) { return P + (P >> 4) + 1; }

// position (unpadded smem index) of frequency k after the forward transform, and its inverse
__host__ __device__ inline int pos_of_freq(const Plan& pl, int k)
{
    int pos = 0, lgM = pl.lgP;
    for (int s = 0; s < pl.nstages; ++s) {
        lgM -= pl.lgR[s];
        pos += (k & ((1 << pl.lgR[s]) - 1)) << lgM;
        k >>= pl.lgR[s];
    }
    return pos;
}
__host__ __device__ inline int freq_of_pos(const Plan& pl, int pos)
{
    int k = 0, lgM = pl.lgP, sh = 0;
    for (int s = 0; s < pl.nstages; ++s) {
        lgM -= pl.lgR[s];
        k += ((pos >> lgM) & ((1 << pl.lgR[s]) - 1)) << sh;
        sh += pl.lgR[s];
    }
    return k;
}

inline Plan make_plan(int lgP)
{
    Plan p{}; p.lgP = lgP; p.nstages = 0;
    int left = lgP;
    while (left >= 4) { p.lgR[p.nstages++] = 4; left -= 4; }
    if (left > 0) p.lgR[p.nstages++] = left;
    return p;
}

#ifdef __CUDACC__

// MMC_FADD2 (default on): a complex add / subtract is ONE packed instruction (sm_100 FADD2: both halves in one issue slot; same
// round-to-nearest results bit for bit).  The FP32 pipe does the same 128 lane results per cycle and SM either way (measured:
// 36.6 against 37.0 T lane results/s), what the packed form saves is issue slots and code size.
#ifndef MMC_FADD2
#define MMC_FADD2 1
#endif
#if MMC_FADD2
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
#else
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x)); }
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) { return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y)); }   // a * conj(b)

// multiply by exp(-/+ 2 pi i k / N) for compile-time k < N/2, N <= 32 (INV: conjugate root)
// P2: the generic root as two packed instructions (FMUL2 + FFMA2 with broadcast scalars; the constants sit in uniform registers)
// instead of two FMUL + two FFMA: the same products and the same fused additions, so the same bits
template <int N, bool INV, bool P2 = false>
__device__ __forceinline__ float2 mul_root(float2 a, int k)
{
    static_assert(N <= 32 && (32 % N) == 0, "mul_root: the root table covers N = 2, 4, 8, 16, 32");
    // cos, sin of 2 pi j / 32, j = 0..15
    constexpr float C[16] = { 1.f, 0.98078528040323044f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
                              0.55557023301960222f, 0.38268343236508977f, 0.19509032201612827f, 0.f,
                              -0.19509032201612827f, -0.38268343236508977f, -0.55557023301960222f, -0.70710678118654752f,
                              -0.83146961230254524f, -0.92387953251128674f, -0.98078528040323044f };
    constexpr float S[16] = { 0.f, 0.19509032201612827f, 0.38268343236508977f, 0.55557023301960222f, 0.70710678118654752f,
                              0.83146961230254524f, 0.92387953251128674f, 0.98078528040323044f, 1.f,
                              0.98078528040323044f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
                              0.55557023301960222f, 0.38268343236508977f, 0.19509032201612827f };
    const int j = k * (32 / N);                       // 0 <= j < 16
    if (j == 0) return a;
    if (j == 8) return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
    const float c = C[j], s = INV ? S[j] : -S[j];     // root = c + i s
    if constexpr (P2) return __ffma2_rn(make_float2(a.x, a.x), make_float2(c, s), __fmul2_rn(make_float2(a.y, a.y), make_float2(-s, c)));
    else return make_float2(fmaf(a.x, c, -a.y * s), fmaf(a.x, s, a.y * c));
}

// radix-2 DIF network on N registers: natural in, bit-reversed out (X[q] ends in x[bitrev(q)])
template <int N, bool INV, bool P2 = false>
__device__ __forceinline__ void dif(float2* x)
{
    if constexpr (N >= 2) {
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float2 a = x[k], b = x[k + N / 2];
            x[k] = cadd(a, b);
            x[k + N / 2] = mul_root<N, INV, P2>(csub(a, b), k);
        }
        dif<N / 2, INV, P2>(x);
        dif<N / 2, INV, P2>(x + N / 2);
    }
}
// radix-2 DIT network: bit-reversed in, natural out
template <int N, bool INV, bool P2 = false>
__device__ __forceinline__ void dit(float2* x)
{
    if constexpr (N >= 2) {
        dit<N / 2, INV, P2>(x);
        dit<N / 2, INV, P2>(x + N / 2);
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float2 a = x[k], b = mul_root<N, INV, P2>(x[k + N / 2], k);
            x[k] = cadd(a, b);
            x[k + N / 2] = csub(a, b);
        }
    }
}
template <int N> __host__ __device__ constexpr int bitrev(int q)
{
    int r = 0;
    for (int b = 1, t = N >> 1; b < N; b <<= 1, t >>= 1) if (q & b) r |= t;
    return r;
}

// One forward stage of radix R = 2^LGR on `nbatch` transforms of length 2^lgP stored at s + b * bstride (padded
// indexing); lgL = log2 of the current block length.  tw[k] = exp(-2 pi i k / 2^lgTw), lgTw >= lgL.
template <int LGR>
__device__ __forceinline__ void stage_fwd(float2* s, int lgP, int lgL, int nbatch, int bstride,
                                          const float2* __restrict__ tw, int lgTw, int tid, int nthreads)
{
    constexpr int R = 1 << LGR;
    const int lgM = lgL - LGR, M = 1 << lgM, lgW = lgP - LGR;
    const int total = nbatch << lgW;
    for (int w = tid; w < total; w += nthreads) {
        const int b = w >> lgW, i = w & ((1 << lgW) - 1);
        const int n = i & (M - 1), i0 = ((i >> lgM) << lgL) + n;
        float2* base = s + b * bstride;
        float2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = base[pad(i0 + (r << lgM))];
        dif<R, false>(x);
#pragma unroll
        for (int q = 0; q < R; ++q) {
            float2 y = x[bitrev<R>(q)];
            if (q > 0 && lgM > 0) y = cmul(y, __ldg(tw + ((n * q) << (lgTw - lgL))));
            base[pad(i0 + (q << lgM))] = y;
        }
    }
}
// The mirror: undoes stage_fwd up to the factor R.
template <int LGR>
__device__ __forceinline__ void stage_inv(float2* s, int lgP, int lgL, int nbatch, int bstride,
                                          const float2* __restrict__ tw, int lgTw, int tid, int nthreads)
{
    constexpr int R = 1 << LGR;
    const int lgM = lgL - LGR, M = 1 << lgM, lgW = lgP - LGR;
    const int total = nbatch << lgW;
    for (int w = tid; w < total; w += nthreads) {
        const int b = w >> lgW, i = w & ((1 << lgW) - 1);
        const int n = i & (M - 1), i0 = ((i >> lgM) << lgL) + n;
        float2* base = s + b * bstride;
        float2 x[R];
#pragma unroll
        for (int q = 0; q < R; ++q) {
            float2 y = base[pad(i0 + (q << lgM))];
            if (q > 0 && lgM > 0) y = cmulc(y, __ldg(tw + ((n * q) << (lgTw - lgL))));
            x[bitrev<R>(q)] = y;
        }
        dit<R, true>(x);
#pragma unroll
        for (int r = 0; r < R; ++r) base[pad(i0 + (r << lgM))] = x[r];
    }
}

template <bool INVERSE>
__device__ __forceinline__ void run_stage(int lgR, float2* s, int lgP, int lgL, int nbatch, int bstride,
                                          const float2* __restrict__ tw, int lgTw, int tid, int nthreads)
{
    if (INVERSE) {
        switch (lgR) {
            case 4: stage_inv<4>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            case 3: stage_inv<3>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            case 2: stage_inv<2>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            default: stage_inv<1>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
        }
    } else {
        switch (lgR) {
            case 4: stage_fwd<4>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            case 3: stage_fwd<3>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            case 2: stage_fwd<2>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
            default: stage_fwd<1>(s, lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads); break;
        }
    }
}

// Whole transforms (block-wide; ends with a __syncthreads so the caller may read any element).
__device__ __forceinline__ void fft_forward(const Plan& pl, float2* s, int nbatch, int bstride,
                                            const float2* __restrict__ tw, int lgTw, int tid, int nthreads)
{
    int lgL = pl.lgP;
    for (int st = 0; st < pl.nstages; ++st) {
        run_stage<false>(pl.lgR[st], s, pl.lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads);
        lgL -= pl.lgR[st];
        __syncthreads();
    }
}
__device__ __forceinline__ void fft_inverse(const Plan& pl, float2* s, int nbatch, int bstride,
                                            const float2* __restrict__ tw, int lgTw, int tid, int nthreads)
{
    int lgL = 0;
    for (int st = pl.nstages - 1; st >= 0; --st) {
        lgL += pl.lgR[st];
        run_stage<true>(pl.lgR[st], s, pl.lgP, lgL, nbatch, bstride, tw, lgTw, tid, nthreads);
        __syncthreads();
    }
}

#endif  // __CUDACC__

}  // namespace fft
}  // namespace mmc

#endif
