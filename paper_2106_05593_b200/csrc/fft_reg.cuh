// fft_reg.cuh -- register-resident power-of-two complex FFTs for the demag convolution (demag.cu), lengths 2^8 .. 2^12.
//
// Every thread keeps 16 points of one transform in registers; a transform of length N = 16 * 16 * R3 (R3 = N/256 in
// {1, 2, 4, 8, 16}) is two radix-16 steps and one radix-R3 step with two exchanges through shared memory in between.
// All lengths, strides and radices are template parameters, so every shared-memory access is "per-thread base +
// immediate" and the butterflies are straight-line code; the twiddles of a thread are the powers of one root per
// stage (w_N^tid, w_T^(tid>>4)), formed in registers, so no twiddle table is read.  T = N/16 threads work on one transform.
//
// Forward (decimation in frequency), thread `tid` of the transform:
//   in   v[n1] = x[tid + n1*T]                                  (HALF: x[n] = 0 for n >= N/2 is folded at compile time)
//   1    radix-16 over n1, twiddle w_N^(tid*q1)                 -> s1[q1*(T+1) + tid]
//   2    thread = (u = tid>>4, q1 = tid&15): radix-16 over t1 of s1[q1*(T+1) + t1*R3 + u], twiddle w_T^(u*q2)
//                                                               -> s2[u*272 + 17*q1 + q2]
//   3    pairs p = tid + i*T (i < 16/R3), p = 16*q1 + q2: radix-R3 over u of s2[u*272 + p + (p>>4)]
//   out  v[i*R3 + q3] = X[q1 + 16*q2 + 256*q3]
// The output order is whatever falls out (freq_of_slot below); the convolution multiplies in that order (the tensor
// spectrum is stored permuted), and the inverse transform is the exact mirror, so no reordering pass exists.
// The paddings (T+1, 17, 272) make every exchange access hit distinct bank pairs within a half-warp.
#ifndef MMC_FFT_REG_CUH_
#define MMC_FFT_REG_CUH_

#include "fft_smem.cuh"

namespace mmc {
namespace fftr {

constexpr int kMinLg = 8, kMaxLg = 12;

template <int LGN>
struct Shape {
    static constexpr int N = 1 << LGN, T = N / 16, R3 = N / 256, NI = 16 / R3;
    static constexpr int U = 272;                                  // row stride of exchange buffer 2
    static constexpr int S1 = 16 * (T + 1);                        // float2 elements of exchange buffer 1
    static constexpr int S2 = R3 > 1 ? R3 * U : 0;                 // ... and 2
    static constexpr int SMEM = S1 + S2;                           // per transform group
    static constexpr int G = T >= 128 ? 1 : 128 / T;               // transforms side by side in one CTA
};

// frequency held by register slot e of thread tid after forward<LGN>
__host__ __device__ inline int freq_of_slot(int lgN, int tid, int e)
{
    const int N = 1 << lgN, T = N / 16, R3 = N / 256;
    if (R3 == 1) return tid + 16 * e;
    const int i = e / R3, q3 = e % R3, p = tid + i * T;
    return (p >> 4) + 16 * (p & 15) + 256 * q3;
}

#ifdef __CUDACC__

// exp(-2 pi i num / den), |num/den| <= 1: sincospif is exact in its range reduction and ~1 ulp
__device__ __forceinline__ float2 root(int num, int den)
{
    float sn, cs;
    sincospif(-2.f * (float)num / (float)den, &sn, &cs);      // num/den is exact for den a power of two, num < 2^24
    return make_float2(cs, sn);
}
// pw[q-1] = w^q, q = 1..15, by a product tree of depth <= 4 (a few ulp): the stage twiddles of a thread are the
// powers of ONE root (w_N^tid, w_T^u), so no twiddle table is read anywhere
__device__ __forceinline__ void powers15(float2 w, float2 (&pw)[15])
{
    pw[0] = w;
    pw[1] = fft::cmul(w, w);
    pw[2] = fft::cmul(pw[1], w);
    pw[3] = fft::cmul(pw[1], pw[1]);
#pragma unroll
    for (int q = 0; q < 3; ++q) pw[4 + q] = fft::cmul(pw[3], pw[q]);
    pw[7] = fft::cmul(pw[3], pw[3]);
#pragma unroll
    for (int q = 0; q < 7; ++q) pw[8 + q] = fft::cmul(pw[7], pw[q]);
}

// Stage twiddles of one thread, either way:
//   computed: the powers of w1 = w_N^tid and w2 = w_T^(tid>>4) (kernels whose L1 is taken by shared memory)
//   table:    t1[(q-1)*T + tid] = w_N^(tid q), t2[(q-1)*T + tid] = w_T^((tid>>4) q), q = 1..15, L1-resident
struct Twiddles { float2 w1, w2; const float2* t1; const float2* t2; };

__global__ void twiddle_tables_kernel(float2* t1, float2* t2, int lgN)
{
    const int N = 1 << lgN, T = N / 16;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < 15 * T; idx += gridDim.x * blockDim.x) {
        const int q = idx / T + 1, t = idx % T;
        double s, c;
        sincospi(-2.0 * (double)(t * q) / (double)N, &s, &c);
        t1[idx] = make_float2((float)c, (float)s);
        sincospi(-2.0 * (double)((t >> 4) * q) / (double)T, &s, &c);
        t2[idx] = make_float2((float)c, (float)s);
    }
}

// TABLE: 0 = computed in registers, 1 = table in global memory read through L1 (__ldg), 2 = table in shared memory
// (kernels whose shared memory leaves no L1; the short latency also lets the compiler fetch each twiddle where it is used
// instead of holding 15 of them in registers)
template <int T, int TABLE>
__device__ __forceinline__ void stage_twiddles(float2 w, const float2* __restrict__ tab, int tid, float2 (&pw)[15])
{
    if (TABLE == 1) {
#pragma unroll
        for (int q = 0; q < 15; ++q) pw[q] = __ldg(tab + q * T + tid);
    } else if (TABLE == 2) {
#pragma unroll
        for (int q = 0; q < 15; ++q) pw[q] = tab[q * T + tid];
    } else {
        powers15(w, pw);
    }
}

// Barrier of the threads that share one transform's exchange buffers: the whole CTA (default), or a named barrier of one
// warp-aligned thread group (several independent transforms in one CTA that should not wait for one another).
struct BlockSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
struct GroupSync {
    int id, n;                                        // barrier 1..15, threads (a multiple of 32)
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
};

template <int LGN, bool HALF, int TABLE, class Sync = BlockSync, bool P2 = false>
__device__ __forceinline__ void forward(float2 (&v)[16], float2* __restrict__ s1, float2* __restrict__ s2,
                                        const Twiddles& tw, int tid, const Sync& sync = Sync())
{
    using S = Shape<LGN>;
    constexpr int T = S::T, R3 = S::R3;
    if (HALF) {                                   // first butterfly level with a zero upper half
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k + 8] = fft::mul_root<16, false, P2>(v[k], k);
        fft::dif<8, false, P2>(v); fft::dif<8, false, P2>(v + 8);
    } else {
        fft::dif<16, false, P2>(v);
    }
    {
        float2 pw[15];
        stage_twiddles<T, TABLE>(tw.w1, tw.t1, tid, pw);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float2 y = v[fft::bitrev<16>(q)];
            if (q > 0) y = fft::cmul(y, pw[q - 1]);
            s1[q * (T + 1) + tid] = y;
        }
    }
    float2 pw2[15];                               // requested before the barrier: the registers of v are free here
    if constexpr (R3 > 1 && TABLE != 2) stage_twiddles<T, TABLE>(tw.w2, tw.t2, tid, pw2);
    sync();
    const int u = tid >> 4, q1 = tid & 15;
    {
        const float2* r1 = s1 + q1 * (T + 1) + u;
#pragma unroll
        for (int t1 = 0; t1 < 16; ++t1) v[t1] = r1[t1 * R3];
    }
    fft::dif<16, false, P2>(v);
    if constexpr (R3 > 1) {
        float2* d2 = s2 + u * S::U + 17 * q1;
        if constexpr (TABLE == 2) stage_twiddles<T, TABLE>(tw.w2, tw.t2, tid, pw2);      // shared-memory table: fetched where it is used
        float2 (&pw)[15] = pw2;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float2 y = v[fft::bitrev<16>(q)];
            if (q > 0) y = fft::cmul(y, pw[q - 1]);
            d2[q] = y;
        }
        sync();
        const float2* r2 = s2 + tid + (tid >> 4);
#pragma unroll
        for (int i = 0; i < S::NI; ++i) {
            float2 x[R3];
#pragma unroll
            for (int uu = 0; uu < R3; ++uu) x[uu] = r2[uu * S::U + i * (T + R3)];
            fft::dif<R3, false, P2>(x);
#pragma unroll
            for (int q = 0; q < R3; ++q) v[i * R3 + q] = x[fft::bitrev<R3>(q)];
        }
    } else {
        float2 x[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = v[fft::bitrev<16>(q)];
#pragma unroll
        for (int q = 0; q < 16; ++q) v[q] = x[q];
        sync();                          // buffer 1 was read last: the next transform may overwrite it
    }
}

// the mirror: v[e] = Y[freq_of_slot(tid, e)] on entry, v[n1] = N * y[tid + n1*T] on exit
template <int LGN, int TABLE, class Sync = BlockSync, bool P2 = false>
__device__ __forceinline__ void inverse(float2 (&v)[16], float2* __restrict__ s1, float2* __restrict__ s2,
                                        const Twiddles& tw, int tid, const Sync& sync = Sync())
{
    using S = Shape<LGN>;
    constexpr int T = S::T, R3 = S::R3;
    const int u = tid >> 4, q1 = tid & 15;
    float2 x16[16];
    if constexpr (R3 > 1) {
        float2* d2 = s2 + tid + (tid >> 4);
#pragma unroll
        for (int i = 0; i < S::NI; ++i) {
            float2 x[R3];
#pragma unroll
            for (int q = 0; q < R3; ++q) x[fft::bitrev<R3>(q)] = v[i * R3 + q];
            fft::dit<R3, true, P2>(x);
#pragma unroll
            for (int uu = 0; uu < R3; ++uu) d2[uu * S::U + i * (T + R3)] = x[uu];
        }
        float2 pw[15];
        if constexpr (TABLE != 2) stage_twiddles<T, TABLE>(tw.w2, tw.t2, tid, pw);
        sync();
        if constexpr (TABLE == 2) stage_twiddles<T, TABLE>(tw.w2, tw.t2, tid, pw);
        const float2* r2 = s2 + u * S::U + 17 * q1;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float2 y = r2[q];
            if (q > 0) y = fft::cmulc(y, pw[q - 1]);
            x16[fft::bitrev<16>(q)] = y;
        }
    } else {
#pragma unroll
        for (int q = 0; q < 16; ++q) x16[fft::bitrev<16>(q)] = v[q];
    }
    fft::dit<16, true, P2>(x16);
    {
        float2* d1 = s1 + q1 * (T + 1) + u;
#pragma unroll
        for (int t1 = 0; t1 < 16; ++t1) d1[t1 * R3] = x16[t1];
    }
    {
        float2 pw[15];
        if constexpr (TABLE != 2) stage_twiddles<T, TABLE>(tw.w1, tw.t1, tid, pw);
        sync();
        if constexpr (TABLE == 2) stage_twiddles<T, TABLE>(tw.w1, tw.t1, tid, pw);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            float2 y = s1[q * (T + 1) + tid];
            if (q > 0) y = fft::cmulc(y, pw[q - 1]);
            v[fft::bitrev<16>(q)] = y;
        }
    }
    fft::dit<16, true, P2>(v);
    if constexpr (R3 == 1) sync();       // as in forward
}

// ---- asynchronous bulk copies global -> shared, completion on an mbarrier (cp.async.bulk: the TMA unit moves the bytes,
// no thread waits on a register) -------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned arrivals)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(arrivals) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of asynchronous copies to come
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// bytes: a multiple of 16; dst and src 16-byte aligned
__device__ __forceinline__ void bulk_copy_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}

// Slot bookkeeping for kernels that need to know which frequency a register holds (demag.cu rows kernels):
// freq_of_slot(tid, e) = kbase(tid) + kconst(e); its padded natural-order index k + (k >> 4) = pbase(tid) + pconst(e).
template <int LGN> __device__ __forceinline__ int kbase(int tid) { return Shape<LGN>::R3 == 1 ? tid : (tid >> 4) + 16 * (tid & 15); }
template <int LGN> __device__ __forceinline__ int pbase(int tid) { return Shape<LGN>::R3 == 1 ? tid : (tid >> 4) + 17 * (tid & 15); }
template <int LGN> __host__ __device__ constexpr int kconst(int e)
{
    return Shape<LGN>::R3 == 1 ? 16 * e : (e / Shape<LGN>::R3) * Shape<LGN>::R3 + 256 * (e % Shape<LGN>::R3);
}
template <int LGN> __host__ __device__ constexpr int pconst(int e)
{
    return Shape<LGN>::R3 == 1 ? 17 * e : (e / Shape<LGN>::R3) * Shape<LGN>::R3 + 272 * (e % Shape<LGN>::R3);
}
// low nibble of the frequency is non-zero (decides the padded index of the mirror frequency N - k)
template <int LGN> __device__ __forceinline__ bool lo_nonzero(int tid, int e)
{
    return Shape<LGN>::R3 == 1 ? tid > 0 : (e / Shape<LGN>::R3 > 0 || tid >= 16);
}

#endif  // __CUDACC__

}  // namespace fftr
}  // namespace mmc

#endif
