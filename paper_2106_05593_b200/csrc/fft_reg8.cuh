// fft_reg8.cuh -- register-resident power-of-two complex FFTs with EIGHT points per thread, lengths 2^10 .. 2^12, for the
// columns kernel of the demag convolution on several layers (demag.cu, columns8_kernel).
//
// Why a second shape beside fft_reg.cuh (16 points per thread): the columns kernel keeps all three components of a column in
// registers from the forward transforms through the tensor product into the inverse transforms.  At 16 points per thread that
// is 96 data registers, 168 in all, twelve warps per SM.  At 8 points per thread it is 48 data registers and twice the threads
// per column: more warps to hide the same latencies, for one more exchange per transform.
//
// N = 8 * 8 * 8 * T3 (T3 = N/512 in {2, 4, 8}), T = N/8 threads per transform, forward = decimation in frequency:
//   in   v[n1] = x[tid + n1*T]                                      (HALF: x[n] = 0 for n >= N/2, folded at compile time)
//   A    radix-8 over n1, twiddle w_N^(tid*q1)                      -> X1[q1*T + tid]
//   B    thread = (q1 = tid / T2, u = tid % T2), T2 = N/64: radix-8 over t1 of X1[q1*T + u + t1*T2], twiddle w_T^(u*q2)
//                                                                   -> X2[(8*q1 + q2)*RS2 + u]
//   C    thread = (s = tid / T3, r = tid % T3), s = 8*q1 + q2: radix-8 over u1 of X2[s*RS2 + r + u1*T3], twiddle w_T2^(r*q3)
//                                                                   -> X3[r*RS3 + s + 64*q3]
//   D    sub-problems p = tid + i*T (i < 8/T3), p = s + 64*q3: radix-T3 over r of X3[r*RS3 + p]
//   out  v[i*T3 + q4] = X[q1 + 8*q2 + 64*q3 + 512*q4]
// The inverse is the exact mirror (decimation in time, conjugate twiddles), unnormalised.  The output order is whatever falls
// out (freq_of_slot8); the tensor spectrum is stored in that order.  Row strides RS2 = T2 + T3 and RS3 = 512 + 16/T3 make every
// 64-bit access of a half-warp hit 16 distinct bank pairs in all three exchanges.
// Exchange buffers: X1 and X3 live in buffer `bx`, X2 in `by`; a transform ends READING bx, so the next transform of the same
// thread group must be called with the two buffers swapped (it then starts by writing the buffer that was last read before a
// barrier).
#ifndef MMC_FFT_REG8_CUH_
#define MMC_FFT_REG8_CUH_

#include "fft_smem.cuh"

namespace mmc {
namespace fftr8 {

constexpr int kMinLg = 10, kMaxLg = 12;

template <int LGN>
struct Shape {
    static_assert(LGN >= kMinLg && LGN <= kMaxLg, "fftr8: lengths 2^10 .. 2^12");
    static constexpr int N = 1 << LGN, T = N / 8, T2 = N / 64, T3 = N / 512, NI = 8 / T3;
    static constexpr int RS2 = T2 + T3;
    static constexpr int RS3 = 512 + 16 / T3;
    static constexpr int BUF = N + 64 * T3;            // float2 per exchange buffer: max(8 T, 64 RS2, T3 RS3)
    static constexpr int SMEM = 2 * BUF;
    static constexpr int NTW = 7 * (T + T2 + T3);      // twiddle table entries
};

// frequency held by register slot e of thread tid after forward<LGN>
__host__ __device__ inline int freq_of_slot8(int lgN, int tid, int e)
{
    const int N = 1 << lgN, T = N / 8, T3 = N / 512;
    const int i = e / T3, q4 = e % T3, p = tid + T * i;
    const int s = p & 63, q3 = p >> 6;
    return (s >> 3) + 8 * (s & 7) + 64 * q3 + 512 * q4;
}

#ifdef __CUDACC__

// tw = [ w_N^(t q), q = 1..7, t < T | w_T^(u q), u < T2 | w_T2^(r q), r < T3 ], entry (q-1)*len + index
__global__ void twiddle_tables8_kernel(float2* tw, int lgN)
{
    const int N = 1 << lgN, T = N / 8, T2 = N / 64, T3 = N / 512;
    const int total = 7 * (T + T2 + T3);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        int len, den, off;
        if (idx < 7 * T) { len = T; den = N; off = idx; }
        else if (idx < 7 * (T + T2)) { len = T2; den = T; off = idx - 7 * T; }
        else { len = T3; den = T2; off = idx - 7 * (T + T2); }
        const int q = off / len + 1, t = off % len;
        double s, c;
        sincospi(-2.0 * (double)(t * q) / (double)den, &s, &c);
        tw[idx] = make_float2((float)c, (float)s);
    }
}

template <int LEN>
__device__ __forceinline__ void load7(const float2* __restrict__ tab, int idx, float2 (&pw)[7])
{
#pragma unroll
    for (int q = 0; q < 7; ++q) pw[q] = __ldg(tab + q * LEN + idx);
}

template <int LGN, bool HALF>
__device__ __forceinline__ void forward(float2 (&v)[8], float2* __restrict__ bx, float2* __restrict__ by,
                                        const float2* __restrict__ tw, int tid)
{
    using S = Shape<LGN>;
    constexpr int T = S::T, T2 = S::T2, T3 = S::T3, RS2 = S::RS2, RS3 = S::RS3;
    if (HALF) {                                   // first butterfly level with a zero upper half
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k + 4] = fft::mul_root<8, false>(v[k], k);
        fft::dif<4, false>(v); fft::dif<4, false>(v + 4);
    } else {
        fft::dif<8, false>(v);
    }
    {
        float2 pa[7];
        load7<T>(tw, tid, pa);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float2 y = v[fft::bitrev<8>(q)];
            if (q > 0) y = fft::cmul(y, pa[q - 1]);
            bx[q * T + tid] = y;
        }
    }
    const int q1 = tid / T2, u = tid % T2;
    float2 pb[7];                                 // requested before the barrier
    load7<T2>(tw + 7 * T, u, pb);
    __syncthreads();
    {
        const float2* r1 = bx + q1 * T + u;
#pragma unroll
        for (int t1 = 0; t1 < 8; ++t1) v[t1] = r1[t1 * T2];
    }
    fft::dif<8, false>(v);
    {
        float2* d2 = by + q1 * 8 * RS2 + u;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float2 y = v[fft::bitrev<8>(q)];
            if (q > 0) y = fft::cmul(y, pb[q - 1]);
            d2[q * RS2] = y;
        }
    }
    const int s = tid / T3, r = tid % T3;
    float2 pc[7];
    load7<T3>(tw + 7 * (T + T2), r, pc);
    __syncthreads();
    {
        const float2* r2 = by + s * RS2 + r;
#pragma unroll
        for (int u1 = 0; u1 < 8; ++u1) v[u1] = r2[u1 * T3];
    }
    fft::dif<8, false>(v);
    {
        float2* d3 = bx + r * RS3 + s;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float2 y = v[fft::bitrev<8>(q)];
            if (q > 0) y = fft::cmul(y, pc[q - 1]);
            d3[64 * q] = y;
        }
    }
    __syncthreads();
    {
        const float2* r3 = bx + tid;
#pragma unroll
        for (int i = 0; i < S::NI; ++i) {
            float2 x[T3];
#pragma unroll
            for (int rr = 0; rr < T3; ++rr) x[rr] = r3[rr * RS3 + i * T];
            fft::dif<T3, false>(x);
#pragma unroll
            for (int q = 0; q < T3; ++q) v[i * T3 + q] = x[fft::bitrev<T3>(q)];
        }
    }
}

// the mirror: v[e] = Y[freq_of_slot8(tid, e)] on entry, v[n1] = N * y[tid + n1*T] on exit
template <int LGN>
__device__ __forceinline__ void inverse(float2 (&v)[8], float2* __restrict__ bx, float2* __restrict__ by,
                                        const float2* __restrict__ tw, int tid)
{
    using S = Shape<LGN>;
    constexpr int T = S::T, T2 = S::T2, T3 = S::T3, RS2 = S::RS2, RS3 = S::RS3;
    {
        float2* d3 = bx + tid;
#pragma unroll
        for (int i = 0; i < S::NI; ++i) {
            float2 x[T3];
#pragma unroll
            for (int q = 0; q < T3; ++q) x[fft::bitrev<T3>(q)] = v[i * T3 + q];
            fft::dit<T3, true>(x);
#pragma unroll
            for (int rr = 0; rr < T3; ++rr) d3[rr * RS3 + i * T] = x[rr];
        }
    }
    const int s = tid / T3, r = tid % T3;
    float2 pw[7];
    load7<T3>(tw + 7 * (T + T2), r, pw);
    __syncthreads();
    {
        const float2* r3 = bx + r * RS3 + s;
        float2 x[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float2 y = r3[64 * q];
            if (q > 0) y = fft::cmulc(y, pw[q - 1]);
            x[fft::bitrev<8>(q)] = y;
        }
        fft::dit<8, true>(x);
        float2* d2 = by + s * RS2 + r;
#pragma unroll
        for (int u1 = 0; u1 < 8; ++u1) d2[u1 * T3] = x[u1];
    }
    const int q1 = tid / T2, u = tid % T2;
    load7<T2>(tw + 7 * T, u, pw);
    __syncthreads();
    {
        const float2* r2 = by + q1 * 8 * RS2 + u;
        float2 x[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float2 y = r2[q * RS2];
            if (q > 0) y = fft::cmulc(y, pw[q - 1]);
            x[fft::bitrev<8>(q)] = y;
        }
        fft::dit<8, true>(x);
        float2* d1 = bx + q1 * T + u;
#pragma unroll
        for (int t1 = 0; t1 < 8; ++t1) d1[t1 * T2] = x[t1];
    }
    load7<T>(tw, tid, pw);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        float2 y = bx[q * T + tid];
        if (q > 0) y = fft::cmulc(y, pw[q - 1]);
        v[fft::bitrev<8>(q)] = y;
    }
    fft::dit<8, true>(v);
}

#endif  // __CUDACC__

}  // namespace fftr8
}  // namespace mmc

#endif
