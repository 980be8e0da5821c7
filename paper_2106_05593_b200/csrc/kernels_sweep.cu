// kernels_sweep.cu -- the MMC colour pass (PAPER.md:92 steps 1-4, Eq. (5), (7), (10), (11), (14), (15)) for sm_100a.
//
// One thread owns one cell of the active colour.  A warp owns 32 consecutive compact indices of one mesh row of the
// colour-split layout (mmc_internal.h), so every load of the warp is one fully used 128-byte line: the cell's own
// vector and B_d, the same compact index of the other colour's row (one x neighbour), that index +-1 (the other x
// neighbour), and the same compact index of the four adjacent rows (y and z neighbours).  A CTA is a 32 x BY x BZ
// brick of such cells, so most neighbour lines are shared inside the CTA and come from L1.  Few live registers per
// thread (one cell) buy the occupancy that hides the HBM latency; the instruction stream, not the byte stream, is
// the tighter bound of this kernel.
// RNG: one Philox4x32-10 block per cell per sweep keyed by the natural cell index (replayable on the CPU side).
#include <cuda_runtime.h>

#include "mmc_internal.h"

namespace mmc {

// ------------------------------------------------------------------------------------------------ RNG
// Philox4x32-10: round  (c0,c1,c2,c3) <- (mulhi(M1,c2)^c1^k0, mullo(M1,c2), mulhi(M0,c0)^c3^k1, mullo(M0,c0)),
// key schedule k0 += 0x9E3779B9, k1 += 0xBB67AE85.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, unsigned k0, unsigned k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c.x;
        const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c.z;
        c = make_uint4((unsigned)(p1 >> 32) ^ c.y ^ k0, (unsigned)p1, (unsigned)(p0 >> 32) ^ c.w ^ k1, (unsigned)p0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}
// 23-bit uniform strictly inside (0,1): ((x>>9) + 0.5) * 2^-23, exact in fp32.
// (The conversion-free form uint_as_float(0x3f800000 | x>>9) - (1 - 2^-24) gives the same value exactly; measured 2 us slower.)
__device__ __forceinline__ float u01(unsigned x) { return fmaf((float)(x >> 9), 1.1920928955078125e-7f, 5.9604644775390625e-8f); }

// Single-instruction approximations (MUFU), flush-to-zero: inputs here are never denormal (|m|^2 > 0 is checked at
// set_m, u in (0,1)).  Relative error <= 2^-22 each, far inside the stage-1 parity tolerance.
__device__ __forceinline__ float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// the same with one Newton step, y <- y + (y/2)(1 - x y^2): ~1 ulp, for the two normalisations that set |m + dm|
__device__ __forceinline__ float rsqrt_1ulp(float x) { const float y = rsqrt_fast(x); return fmaf(0.5f * y, fmaf(-x * y, y, 1.f), y); }
__device__ __forceinline__ float sqrt_fast(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float ln_fast(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y * 0.693147180559945309f; }

// sin and cos of 2 pi u for u in (0,1): quadrant k = rint(4u), r = 4u - k in [-1/2, 1/2] (exact), Taylor polynomials
// of sin(pi r/2) and cos(pi r/2) (truncation < 3e-8), quadrant fix-up by sign-bit XOR.  No branches, no slow path.
__device__ __forceinline__ void sincos_2pi(float u, float* sn, float* cs)
{
    const float t = 4.f * u;
    const float tr = t + 12582912.f;                   // 1.5 * 2^23: the low mantissa bits now hold rint(t)
    const unsigned k = __float_as_uint(tr);
    const float r = t - (tr - 12582912.f);
    const float r2 = r * r;
    float ps = 1.6044118478736e-4f;                    // (pi/2)^9 / 9!
    ps = fmaf(ps, r2, -4.6817541353187e-3f);           // -(pi/2)^7 / 7!
    ps = fmaf(ps, r2, 7.9692626246167e-2f);            // (pi/2)^5 / 5!
    ps = fmaf(ps, r2, -6.4596409750625e-1f);           // -(pi/2)^3 / 3!
    ps = fmaf(ps, r2, 1.5707963267949f);               // pi/2
    const float s0 = ps * r;
    float pc = 9.1926027483942e-4f;                    // (pi/2)^8 / 8!
    pc = fmaf(pc, r2, -2.0863480763353e-2f);           // -(pi/2)^6 / 6!
    pc = fmaf(pc, r2, 2.5366950790105e-1f);            // (pi/2)^4 / 4!
    pc = fmaf(pc, r2, -1.2337005501362f);              // -(pi/2)^2 / 2!
    const float c0 = fmaf(pc, r2, 1.f);
    const bool swap = (k & 1u) != 0u;
    const float cq = swap ? s0 : c0, sq = swap ? c0 : s0;
    *cs = __uint_as_float(__float_as_uint(cq) ^ (((k + 1u) << 30) & 0x80000000u));   // k = 1, 2: negative
    *sn = __uint_as_float(__float_as_uint(sq) ^ ((k << 30) & 0x80000000u));          // k = 2, 3: negative
}

struct CellCoef {
    float kx, ky, kz, gx, gy, bKq, bzee, c4, sigma, ax, ay, az;
    double mu2;
    float bK1c, bK2c, cub[9], bK2u;    // higher-order anisotropy (only read when CUBIC)
};

// cubic table slots CS_BK1C, CS_BK2C, CS_CUB .. CS_CUB + 8 of a class
__device__ __forceinline__ void load_cubic(const float4* t, CellCoef& cf)
{
    const float4 t3 = __ldg(t), t4 = __ldg(t + 1), t5 = __ldg(t + 2);
    cf.bK1c = t3.x; cf.bK2c = t3.y; cf.cub[0] = t3.z; cf.cub[1] = t3.w;
    cf.cub[2] = t4.x; cf.cub[3] = t4.y; cf.cub[4] = t4.z; cf.cub[5] = t4.w;
    cf.cub[6] = t5.x; cf.cub[7] = t5.y; cf.cub[8] = t5.z; cf.bK2u = t5.w;
}

struct CellResult { float dm[3]; float f, L; float terms[6]; float margin; bool accept; };

// The per-cell body: trial move (O3), dF/kBT (O4), Eq. (5) in the log domain (O5).
//   m      : current vector          S  : sum_d k_d sum_{bonded nb in d}(m_nb - m)   (beta J_d folded into k_d)
//   selfc  : sum_d k_d n_d / 2       dzx, dzy, dxx, dyy : E-W / N-S differences of m_z, m_x, m_y for the DMI vector
//   B      : B_ext + B_d (tesla); TERMS (debug) keeps Zeeman and demag apart for the per-term dump
template <bool DMI, bool TERMS, bool CUBIC>
__device__ __forceinline__ CellResult cell_update(const float m[3], const float S[3], float selfc,
                                                  float dzx, float dzy, float dxx, float dyy,
                                                  const float Bext[3], const float Bd[3],
                                                  const CellCoef& cf, uint4 rnd, float omc)
{
    CellResult r;
    const float u_cos = u01(rnd.x), u_phi = u01(rnd.y), u_len = u01(rnd.z), u_acc = u01(rnd.w);
    const float l2 = fmaf(m[0], m[0], fmaf(m[1], m[1], m[2] * m[2]));
    const float iL = rsqrt_1ulp(l2), L = l2 * iL;
    const float n0 = m[0] * iL, n1 = m[1] * iL, n2 = m[2] * iL;
    // tangent frame (O3): a = axis of the smallest |m_a| (raw components, ties -> lowest index), t1 = e_a x n / |.|,
    // t2 = n x t1.  In the cyclic order (a,b,c) starting at that axis: t1 = (0,-n_c,n_b) it, t2 = (n_b^2+n_c^2,
    // -n_a n_b, -n_a n_c) it with it = 1/sqrt(n_b^2+n_c^2); a cyclic relabelling keeps the handedness.
    const float a0 = fabsf(m[0]), a1 = fabsf(m[1]), a2 = fabsf(m[2]);
    const bool sel1 = a1 < a0;                         // axis 1 beats axis 0
    const bool sel2 = a2 < (sel1 ? a1 : a0);           // axis 2 beats the better of 0, 1
    const float na = sel2 ? n2 : (sel1 ? n1 : n0);
    const float nb = sel2 ? n0 : (sel1 ? n2 : n1);
    const float nc = sel2 ? n1 : (sel1 ? n0 : n2);
    const float p2 = fmaf(nb, nb, nc * nc);
    const float it = rsqrt_1ulp(p2);
    const float w = u_cos * omc;                       // 1 - cos(theta), uniform on the cap
    const float st = sqrt_fast(w * (2.f - w));
    float sp, cp;
    sincos_2pi(u_phi, &sp, &cp);
    const float ca = st * cp * it, sa = st * sp * it;  // coefficients of the un-normalised t1, t2
    // dn = ca (0,-nc,nb) + sa (p2, -na nb, -na nc) - w (na,nb,nc), in the (a,b,c) order
    const float da = fmaf(sa, p2, -w * na);
    const float db = fmaf(-ca, nc, fmaf(-sa * na, nb, -w * nb));
    const float dc = fmaf(ca, nb, fmaf(-sa * na, nc, -w * nc));
    const float dn0 = sel2 ? db : (sel1 ? dc : da);
    const float dn1 = sel2 ? dc : (sel1 ? da : db);
    const float dn2 = sel2 ? da : (sel1 ? db : dc);
    const float s = cf.sigma * fmaf(2.f, u_len, -1.f);  // f = 1 + s
    const float f = 1.f + s;
    const float dm0 = L * fmaf(f, dn0, s * n0), dm1 = L * fmaf(f, dn1, s * n1), dm2 = L * fmaf(f, dn2, s * n2);
    r.dm[0] = dm0; r.dm[1] = dm1; r.dm[2] = dm2; r.f = f; r.L = L;
    // exchange: -dm.S + selfc |dm|^2
    const float dmsq = fmaf(dm0, dm0, fmaf(dm1, dm1, dm2 * dm2));
    const float ex = fmaf(selfc, dmsq, -fmaf(dm0, S[0], fmaf(dm1, S[1], dm2 * S[2])));
    // uniaxial anisotropy: -beta V Kq (dm.e)((2m+dm).e)
    const float dme = fmaf(dm0, cf.ax, fmaf(dm1, cf.ay, dm2 * cf.az));
    const float sme = fmaf(fmaf(2.f, m[0], dm0), cf.ax, fmaf(fmaf(2.f, m[1], dm1), cf.ay, fmaf(2.f, m[2], dm2) * cf.az));
    float an = -cf.bKq * dme * sme;
    if (CUBIC) {
        // Eq. (11), second term: V K2(T) [1 - q/me^2]^2 with q = (m.e)^2; its change is -dq (2 (me^2 - q) - dq) K2(T)/me^4,
        // dq = (dm.e)((2m+dm).e); bK2u = beta V K2(T)/me^4, mu2 = me^2 below Tc (bK2u = 0 above)
        {
            const float qe = fmaf(m[0], cf.ax, fmaf(m[1], cf.ay, m[2] * cf.az));
            const float dq = dme * sme;
            an = fmaf(-cf.bK2u * dq, fmaf(2.f, (float)cf.mu2 - qe * qe, -dq), an);
        }
        // Eq. (12) for the directions n and n' = n + dn (the trial vector is L f (n + dn)): squares of the direction cosines
        // A, B, G and their changes dA = d(alpha)(2 alpha + d(alpha)), ...; both invariants as differences without cancellation
        const float al = fmaf(n0, cf.cub[0], fmaf(n1, cf.cub[1], n2 * cf.cub[2]));
        const float be = fmaf(n0, cf.cub[3], fmaf(n1, cf.cub[4], n2 * cf.cub[5]));
        const float ga = fmaf(n0, cf.cub[6], fmaf(n1, cf.cub[7], n2 * cf.cub[8]));
        const float dal = fmaf(dn0, cf.cub[0], fmaf(dn1, cf.cub[1], dn2 * cf.cub[2]));
        const float dbe = fmaf(dn0, cf.cub[3], fmaf(dn1, cf.cub[4], dn2 * cf.cub[5]));
        const float dga = fmaf(dn0, cf.cub[6], fmaf(dn1, cf.cub[7], dn2 * cf.cub[8]));
        const float A = al * al, B = be * be, G = ga * ga;
        const float dA = dal * fmaf(2.f, al, dal), dB = dbe * fmaf(2.f, be, dbe), dG = dga * fmaf(2.f, ga, dga);
        const float Ap = A + dA, Bp = B + dB;
        const float d1 = fmaf(A, dB, fmaf(Bp, dA, fmaf(A, dG, fmaf(G + dG, dA, fmaf(B, dG, (G + dG) * dB)))));
        const float d2 = fmaf(dA * B, G, Ap * fmaf(dB, G, Bp * dG));
        an = fmaf(cf.bK1c, d1, fmaf(cf.bK2c, d2, an));
    }
    // Zeeman + demag: -beta V Ms0 dm.(B_ext + B_d)
    float zee, dem;
    if (TERMS) {
        zee = -cf.bzee * fmaf(dm0, Bext[0], fmaf(dm1, Bext[1], dm2 * Bext[2]));
        dem = -cf.bzee * fmaf(dm0, Bd[0], fmaf(dm1, Bd[1], dm2 * Bd[2]));
    } else {
        zee = -cf.bzee * fmaf(dm0, Bext[0] + Bd[0], fmaf(dm1, Bext[1] + Bd[1], dm2 * (Bext[2] + Bd[2])));
        dem = 0.f;
    }
    // interfacial DMI: -2 beta D0 V dm.G, G = 1/2(-dzx/dx, -dzy/dy, dxx/dx + dyy/dy); gx = beta D0 V/dx
    float dmi = 0.f;
    if (DMI) dmi = fmaf(dm0, cf.gx * dzx, fmaf(dm1, cf.gy * dzy, -dm2 * fmaf(cf.gx, dxx, cf.gy * dyy)));
    // longitudinal: dl2 c4 (2 (l2 - mu2) + dl2), dl2 = |m'|^2 - |m|^2 = l2 s (2 + s) from the length factor (O3:
    // |m'| = f |m|; the unit vectors above are normalised to ~1 ulp so that the stored m + dm honours this to a
    // few 1e-7).  The bracket l2 - mu2 cancels 2-3 digits below Tc, so it is formed in fp64 from the exact squares
    // of the stored fp32 components.
    const double l2d = fma((double)m[0], (double)m[0], fma((double)m[1], (double)m[1], (double)m[2] * (double)m[2]));
    const float dev = (float)(l2d - cf.mu2);
    const float dl2 = l2 * (s * (2.f + s));
    const float lng = dl2 * cf.c4 * fmaf(2.f, dev, dl2);
    const float dF = ((ex + an) + (zee + dem)) + (dmi + lng);
    // Eq. (5): accept iff ln u < 4 ln f - dF
    r.margin = ln_fast(u_acc) - 4.f * ln_fast(f) + dF;
    r.accept = r.margin < 0.f;
    if (TERMS) { r.terms[0] = ex; r.terms[1] = an; r.terms[2] = zee; r.terms[3] = dmi; r.terms[4] = dem; r.terms[5] = lng; }
    return r;
}

// ---- S10: acceptance counters and running sums.  Thread: counts and the final vectors of its cells.  Warp: integer REDUX
// of the packed counts and of the fixed-point sums (kSumScale = 2^22; a warp's <= 64 cells stay far inside int32).  Block:
// 32-bit shared atomics by lane 0 (two accumulators per sum, for even and odd warps: each collects <= 256 cells, so it
// cannot overflow for |m| < 2); the last warp to sign in on the arrival counter flushes the block's totals with six global
// 64-bit atomics.  No barrier after the update, so early warps retire at once.  Integer arithmetic throughout: exact,
// order-independent, deterministic.
// (Measured on a cfg 4 pass of 57 us: this tail costs about 10 us.  Alternatives measured and dropped: 64-bit shared atomics
// (a CAS loop: +12 us), per-warp partials in plain shared stores summed by the last warp (+19 us), a block barrier + warp 0
// (+16 us with 512-thread CTAs).)
struct PassTailSmem { unsigned cnt[2]; unsigned sum[2][4]; unsigned arrived; };

__device__ __forceinline__ void pass_tail_init(PassTailSmem& sm)
{
    const int tlin = threadIdx.x + 32 * (threadIdx.y + blockDim.y * threadIdx.z);
    if (tlin < 2) sm.cnt[tlin] = 0u;
    if (tlin >= 2 && tlin < 10) (&sm.sum[0][0])[tlin - 2] = 0u;
    if (tlin == 10) sm.arrived = 0u;
    __syncthreads();                                  // the only block barrier: all warps are still in step here
}

__device__ __forceinline__ void pass_tail(const SweepArgs& a, PassTailSmem& sm, unsigned n_acc, unsigned n_tri,
                                          float fs0, float fs1, float fs2, float fs3, int warps)
{
    const bool want_sums = a.run_sums != nullptr;
    const unsigned cnt = __reduce_add_sync(0xffffffffu, n_acc | (n_tri << 16));      // <= 64 each: no carry between the halves
    int i0 = 0, i1 = 0, i2 = 0, i3 = 0;
    if (want_sums) {
        i0 = __reduce_add_sync(0xffffffffu, __float2int_rn(fs0 * kSumScale));
        i1 = __reduce_add_sync(0xffffffffu, __float2int_rn(fs1 * kSumScale));
        i2 = __reduce_add_sync(0xffffffffu, __float2int_rn(fs2 * kSumScale));
        i3 = __reduce_add_sync(0xffffffffu, __float2int_rn(fs3 * kSumScale));
    }
    if (threadIdx.x == 0) {
        if (cnt >> 16) {
            const int par = (threadIdx.y + blockDim.y * threadIdx.z) & 1;
            atomicAdd(&sm.cnt[0], cnt & 0xffffu);
            atomicAdd(&sm.cnt[1], cnt >> 16);
            if (want_sums) {
                atomicAdd(&sm.sum[par][0], (unsigned)i0); atomicAdd(&sm.sum[par][1], (unsigned)i1);
                atomicAdd(&sm.sum[par][2], (unsigned)i2); atomicAdd(&sm.sum[par][3], (unsigned)i3);
            }
        }
        __threadfence_block();
        if (atomicAdd(&sm.arrived, 1u) == (unsigned)(warps - 1)) {      // last warp of the block
            __threadfence_block();
            const unsigned tc = atomicAdd(&sm.cnt[1], 0u);
            if (tc) {
                atomicAdd(&a.ctl->win_trials, (unsigned long long)tc);
                const unsigned ac = atomicAdd(&sm.cnt[0], 0u);
                if (ac) atomicAdd(&a.ctl->win_accepted, (unsigned long long)ac);
                if (want_sums)                         // sign-extend the two 32-bit two's-complement halves
                    for (int t = 0; t < 4; ++t)
                        atomicAdd(&a.run_sums[t], (unsigned long long)((long long)(int)atomicAdd(&sm.sum[0][t], 0u) +
                                                                       (long long)(int)atomicAdd(&sm.sum[1][t], 0u)));
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ the pass
// blockDim = (32, BY, BZ), kPassThreads = 512 threads (measured on cfg 4 / cfg 5: 128 threads 110 / 100 us per pass,
// 256: 69 / 59, 512: 65 / 52, 1024: 68 / 55: the larger brick shares more neighbour rows through L1);
// grid = (ceil(hxr/32), ceil(ny/BY), ceil(nz/BZ)).
// Running sums of the sweep's final vectors are kept in fixed point (kSumScale), so that they can be reduced with
// integer warp reductions and integer atomics: exact, order-independent and therefore deterministic.
#ifndef MMC_PASS_THREADS
#define MMC_PASS_THREADS 512
#endif
constexpr int kPassThreads = MMC_PASS_THREADS;      // CTA = 32 x BY x BZ brick of this many cells
// coherent load for the persistent single-CTA kernel, whose passes read what earlier passes of the same launch wrote;
// read-only path otherwise
template <bool COHERENT> __device__ __forceinline__ float ldc(const float* p) { return COHERENT ? __ldcg(p) : __ldg(p); }   // .cg: from L2, never a stale line

// One cell of the active colour: compact index q of row (j, k).  The body of the one-cell-per-thread pass.
template <unsigned F, bool DEBUG, bool COHERENT>
__device__ __forceinline__ void pass_one_cell(const SweepArgs& a, int col, int q, int j, int k, unsigned long long sweep, float omc,
                                              bool& active, bool& accept, float& fs0, float& fs1, float& fs2, float& fs3)
{
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DMI = (F & F_DMI) != 0, DEMAG = (F & F_DEMAG) != 0, DENSE = (F & F_DENSE) != 0, CUBIC = (F & F_CUBIC) != 0;
    const int nx = a.g.nx, ny = a.g.ny, nz = a.g.nz, hx = a.g.hx;
    const unsigned pbc = a.g.pbc;
    const int s = ((j + k) & 1) ^ col;               // active cells of this row sit at i = 2q + s
    const int i = 2 * q + s;
    active = i < nx && j < ny && k < nz;
    accept = false;
    fs0 = fs1 = fs2 = fs3 = 0.f;                      // the cell's final vector and length (running sums)

    // 32-bit element offsets: mmc_create guarantees 2 H < 2^31
    const unsigned H = (unsigned)a.g.H;
    const int row = k * ny + j;
    const unsigned rq = (unsigned)row * hx + q;
    const unsigned ownb = (unsigned)col * H + rq;
    unsigned mb = 0x7fu, cls = 0u;
    if (active) {
        if (PERCELL) { const unsigned w = __ldg(a.cw + ownb); mb = w & 0x7fu; cls = w >> 7; }
        else if (MASK) mb = __ldg(a.mask + ownb);
        // DENSE (no empty cell in the mesh): the vector loads below do not have to wait for this word to arrive
        if (!DENSE && (MASK || PERCELL) && !(mb & 0x40u)) active = false;   // empty cell
    }
    if (active) {
        const int hxr = (nx + 1) >> 1;               // compact length of the real (unpadded) row
        // element deltas from this thread's slot in the other colour's plane to its six neighbours
        // (wrap when periodic, else 0: an out-of-mesh neighbour is never bonded, any valid address will do)
        const int dN = (j + 1 < ny) ? hx : ((pbc & 2u) ? -(ny - 1) * hx : 0);
        const int dS = (j > 0) ? -hx : ((pbc & 2u) ? (ny - 1) * hx : 0);
        // x: s == 0: E at q, W at q-1;  s == 1: W at q, E at q+1
        int dX = s ? 1 : -1;
        if (q + dX < 0) dX = (pbc & 1u) ? hxr - 1 : 0;
        else if (q + dX >= hxr) dX = (pbc & 1u) ? -q : 0;
        int dU = 0, dD = 0;
        if (HASZ) {
            const int lay = ny * hx;
            dU = (k + 1 < nz) ? lay : ((pbc & 4u) ? -(nz - 1) * lay : 0);
            dD = (k > 0) ? -lay : ((pbc & 4u) ? (nz - 1) * lay : 0);
        }
        // 32-bit offsets of the six neighbour slots (all inside [0, 2H)): one add each, one IMAD.WIDE per load
        const unsigned othb = (unsigned)(1 - col) * H + rq;
        const unsigned oX = othb + (unsigned)dX, oN = othb + (unsigned)dN, oS = othb + (unsigned)dS;
        const unsigned oU = othb + (unsigned)dU, oD = othb + (unsigned)dD;
        float m[3], xa[3], xb[3], yn[3], ys[3], zu[3], zd[3], Bd[3] = { 0.f, 0.f, 0.f };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* __restrict__ P = a.m[c];
            m[c] = a.m[c][ownb];
            xa[c] = ldc<COHERENT>(P + othb);
            xb[c] = ldc<COHERENT>(P + oX);
            yn[c] = ldc<COHERENT>(P + oN);
            ys[c] = ldc<COHERENT>(P + oS);
            if (HASZ) { zu[c] = ldc<COHERENT>(P + oU); zd[c] = ldc<COHERENT>(P + oD); }
            if (DEMAG) Bd[c] = __ldg(a.bd[c] + ownb);
        }
        CellCoef cf;
        float kscale = 1.f;
        if (PERCELL) {
            const float4* t = a.table + (kClassFloats / 4) * cls;
            const float4 t0 = __ldg(t), t1 = __ldg(t + 1);
            const float2 t2 = __ldg(reinterpret_cast<const float2*>(t + 2));
            kscale = t0.x; cf.c4 = t0.y;
            cf.mu2 = __hiloint2double(__float_as_int(t0.w), __float_as_int(t0.z));
            cf.bKq = t1.x; cf.bzee = t1.y; cf.sigma = t1.z; cf.ax = t1.w; cf.ay = t2.x; cf.az = t2.y;
            if (CUBIC) load_cubic(a.table_cubic + (kClassFloats / 4) * cls, cf);
        } else {
            cf.bKq = a.coef.bKq; cf.bzee = a.coef.bzee; cf.c4 = a.coef.c4; cf.sigma = a.coef.sigma;
            cf.ax = a.coef.ax; cf.ay = a.coef.ay; cf.az = a.coef.az; cf.mu2 = a.coef.mu2;
            if (CUBIC) { cf.bK1c = a.coef.bK1c; cf.bK2c = a.coef.bK2c; for (int q = 0; q < 9; ++q) cf.cub[q] = a.coef.cub[q]; cf.bK2u = a.coef.bK2u; }
        }
        cf.kx = a.coef.kx * kscale; cf.ky = a.coef.ky * kscale; cf.kz = a.coef.kz * kscale;
        cf.gx = a.coef.gx * kscale; cf.gy = a.coef.gy * kscale;
        // bond weights (1 or 0)
        float bE = 1.f, bW = 1.f, bN = 1.f, bS = 1.f, bU = HASZ ? 1.f : 0.f, bD = HASZ ? 1.f : 0.f;
        if (MASK || PERCELL) {
            bE = (mb & 1u) ? 1.f : 0.f;  bW = (mb & 2u) ? 1.f : 0.f;
            bN = (mb & 4u) ? 1.f : 0.f;  bS = (mb & 8u) ? 1.f : 0.f;
            bU = (mb & 16u) ? 1.f : 0.f; bD = (mb & 32u) ? 1.f : 0.f;
        } else {
            if (nx < 2) { bE = 0.f; bW = 0.f; }
            if (ny < 2) { bN = 0.f; bS = 0.f; }
        }
        float S[3], e[3], wv[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            e[c] = s ? xb[c] : xa[c]; wv[c] = s ? xa[c] : xb[c];
            const float sx = bE * (e[c] - m[c]) + bW * (wv[c] - m[c]);
            const float sy = bN * (yn[c] - m[c]) + bS * (ys[c] - m[c]);
            float acc = fmaf(cf.kx, sx, cf.ky * sy);
            if (HASZ) acc = fmaf(cf.kz, bU * (zu[c] - m[c]) + bD * (zd[c] - m[c]), acc);
            S[c] = acc;
        }
        float selfc = 0.5f * fmaf(cf.kx, bE + bW, cf.ky * (bN + bS));
        if (HASZ) selfc = fmaf(0.5f * cf.kz, bU + bD, selfc);
        float dzx = 0.f, dzy = 0.f, dxx = 0.f, dyy = 0.f;
        if (DMI) {
            dzx = bE * e[2] - bW * wv[2];
            dzy = bN * yn[2] - bS * ys[2];
            dxx = bE * e[0] - bW * wv[0];
            dyy = bN * yn[1] - bS * ys[1];
        }
        const float Bext[3] = { a.coef.Bx, a.coef.By, a.coef.Bz };
        const unsigned cell = (unsigned)row * nx + i;                     // natural cell index (< 2^31)
        const uint4 rnd = philox4x32_10(make_uint4(cell, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi);
        const CellResult r = cell_update<DMI, DEBUG, CUBIC>(m, S, selfc, dzx, dzy, dxx, dyy, Bext, Bd, cf, rnd, omc);
        accept = r.accept;
        fs0 = m[0]; fs1 = m[1]; fs2 = m[2]; fs3 = r.L;
        if (accept) {
            fs0 += r.dm[0]; fs1 += r.dm[1]; fs2 += r.dm[2]; fs3 *= r.f;     // |m'| = f |m| (O3)
            a.m[0][ownb] = fs0; a.m[1][ownb] = fs1; a.m[2][ownb] = fs2;
        }
        if (DEBUG) {
            const size_t c = cell;
            if (a.dbg_dm) { a.dbg_dm[3 * c] = r.dm[0]; a.dbg_dm[3 * c + 1] = r.dm[1]; a.dbg_dm[3 * c + 2] = r.dm[2]; }
            if (a.dbg_terms) for (int t = 0; t < 6; ++t) a.dbg_terms[6 * c + t] = r.terms[t];
            if (a.dbg_margin) a.dbg_margin[c] = r.margin;
            if (a.dbg_acc) a.dbg_acc[c] = r.accept ? 1 : 0;
        }
    }

}

template <unsigned F, bool DEBUG>
__global__ void __launch_bounds__(kPassThreads, DEBUG ? 1 : 1024 / kPassThreads) colour_pass_kernel(const SweepArgs a)
{
    constexpr bool HASZ = (F & F_Z) != 0;
    __shared__ PassTailSmem s_tail;
    pass_tail_init(s_tail);
    const int q = blockIdx.x * 32 + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = HASZ ? blockIdx.z * blockDim.z + threadIdx.z : 0;
    bool active, accept;
    float fs0, fs1, fs2, fs3;
    pass_one_cell<F, DEBUG, false>(a, a.colour, q, j, k, a.ctl->sweep, a.ctl->one_minus_cos_cone, active, accept, fs0, fs1, fs2, fs3);
    pass_tail(a, s_tail, accept ? 1u : 0u, active ? 1u : 0u, fs0, fs1, fs2, fs3, kPassThreads / 32);
}

// ------------------------------------------------------------------------------------------------ the pass, two cells per thread
// The same pass with a thread owning TWO consecutive compact cells of a row (mesh cells i and i + 2): the vectors, B_d and
// class words / masks come as 64-bit loads, the x neighbour between the two cells is loaded once, index arithmetic, bond
// decoding and the reductions are shared.  Used for every non-debug launch unless x is periodic with an odd compact row
// length (then the wrap neighbour of the last cell would not pair up).  blockDim = (32, BY, BZ), 256 threads = a brick of
// 64 x BY x BZ cells of one colour; grid = (ceil(hxr/64), ceil(ny/BY), ceil(nz/BZ)).
constexpr int kPass2Threads = 256;

#ifndef MMC_PASS2_MINB
#define MMC_PASS2_MINB 4      // 64 registers (48 bytes spilled): measured 4 / 3 / 2 CTAs per SM on cfg 4: 57.5 / 61 / 72 us per pass
#endif
template <unsigned F>
__global__ void __launch_bounds__(kPass2Threads, MMC_PASS2_MINB) colour_pass2_kernel(const SweepArgs a)
{
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DMI = (F & F_DMI) != 0, DEMAG = (F & F_DEMAG) != 0, DENSE = (F & F_DENSE) != 0, CUBIC = (F & F_CUBIC) != 0;
    __shared__ PassTailSmem s_tail;
    pass_tail_init(s_tail);

    const int nx = a.g.nx, ny = a.g.ny, nz = a.g.nz, hx = a.g.hx;
    const unsigned pbc = a.g.pbc;
    const int q0 = 2 * (blockIdx.x * 32 + threadIdx.x);           // cells q0 and q0 + 1 of the compact row
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = HASZ ? blockIdx.z * blockDim.z + threadIdx.z : 0;
    const int col = a.colour;
    const int s = ((j + k) & 1) ^ col;                            // active cells of this row sit at i = 2q + s
    const int i0 = 2 * q0 + s;
    const bool inrow = j < ny && k < nz;
    bool act[2] = { inrow && i0 < nx, inrow && i0 + 2 < nx };
    unsigned n_acc = 0u;
    float fs0 = 0.f, fs1 = 0.f, fs2 = 0.f, fs3 = 0.f;

    const unsigned H = (unsigned)a.g.H;
    const int row = k * ny + j;
    const unsigned rq = (unsigned)row * hx + q0;
    const unsigned ownb = (unsigned)col * H + rq;
    unsigned mb[2] = { 0x7fu, 0x7fu }, cls[2] = { 0u, 0u };
    if (act[0]) {                                                 // (cell 1 active implies cell 0 active)
        if (PERCELL) {
            const uint2 w = __ldg(reinterpret_cast<const uint2*>(a.cw + ownb));
            mb[0] = w.x & 0x7fu; cls[0] = w.x >> 7; mb[1] = w.y & 0x7fu; cls[1] = w.y >> 7;
        } else if (MASK) {
            const uchar2 w = __ldg(reinterpret_cast<const uchar2*>(a.mask + ownb));
            mb[0] = w.x; mb[1] = w.y;
        }
        if (!DENSE && (MASK || PERCELL)) { act[0] = act[0] && (mb[0] & 0x40u); act[1] = act[1] && (mb[1] & 0x40u); }
    }
    if (act[0] || act[1]) {
        const int hxr = (nx + 1) >> 1;
        const int dN = (j + 1 < ny) ? hx : ((pbc & 2u) ? -(ny - 1) * hx : 0);
        const int dS = (j > 0) ? -hx : ((pbc & 2u) ? (ny - 1) * hx : 0);
        // the third x neighbour: s == 0: W of cell 0 at q0 - 1; s == 1: E of cell 1 at q0 + 2 (wrap when periodic, else any
        // valid slot: the bond is masked)
        int dX = s ? 2 : -1;
        if (q0 + dX < 0) dX = (pbc & 1u) ? hxr - 1 : 0;
        else if (q0 + dX >= hxr) dX = (pbc & 1u) ? -q0 : 0;
        int dU = 0, dD = 0;
        if (HASZ) {
            const int lay = ny * hx;
            dU = (k + 1 < nz) ? lay : ((pbc & 4u) ? -(nz - 1) * lay : 0);
            dD = (k > 0) ? -lay : ((pbc & 4u) ? (nz - 1) * lay : 0);
        }
        const unsigned othb = (unsigned)(1 - col) * H + rq;
        float2 m2[3], xc[3], yn[3], ys[3], zu[3], zd[3], bd2[3];
        float xs[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* __restrict__ P = a.m[c];
            m2[c] = *reinterpret_cast<const float2*>(a.m[c] + ownb);
            xc[c] = __ldg(reinterpret_cast<const float2*>(P + othb));
            xs[c] = __ldg(P + othb + dX);
            yn[c] = __ldg(reinterpret_cast<const float2*>(P + othb + dN));
            ys[c] = __ldg(reinterpret_cast<const float2*>(P + othb + dS));
            if (HASZ) { zu[c] = __ldg(reinterpret_cast<const float2*>(P + othb + dU)); zd[c] = __ldg(reinterpret_cast<const float2*>(P + othb + dD)); }
            bd2[c] = DEMAG ? __ldg(reinterpret_cast<const float2*>(a.bd[c] + ownb)) : make_float2(0.f, 0.f);
        }
        const unsigned long long sweep = a.ctl->sweep;
        const float omc = a.ctl->one_minus_cos_cone;
        const float Bext[3] = { a.coef.Bx, a.coef.By, a.coef.Bz };
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            if (!act[t]) continue;
            float m[3], e[3], wv[3], N[3], S_[3], U[3], D[3], Bd[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                m[c] = t ? m2[c].y : m2[c].x;
                // s == 0: cell 0: E = xc.x, W = xs; cell 1: E = xc.y, W = xc.x.   s == 1: cell 0: W = xc.x, E = xc.y; cell 1: W = xc.y, E = xs
                if (t == 0) { e[c] = s ? xc[c].y : xc[c].x; wv[c] = s ? xc[c].x : xs[c]; }
                else        { e[c] = s ? xs[c] : xc[c].y;   wv[c] = s ? xc[c].y : xc[c].x; }
                N[c] = t ? yn[c].y : yn[c].x; S_[c] = t ? ys[c].y : ys[c].x;
                if (HASZ) { U[c] = t ? zu[c].y : zu[c].x; D[c] = t ? zd[c].y : zd[c].x; }
                Bd[c] = t ? bd2[c].y : bd2[c].x;
            }
            CellCoef cf;
            float kscale = 1.f;
            if (PERCELL) {
                const float4* tb = a.table + (kClassFloats / 4) * cls[t];
                const float4 t0 = __ldg(tb), t1 = __ldg(tb + 1);
                const float2 t2 = __ldg(reinterpret_cast<const float2*>(tb + 2));
                kscale = t0.x; cf.c4 = t0.y;
                cf.mu2 = __hiloint2double(__float_as_int(t0.w), __float_as_int(t0.z));
                cf.bKq = t1.x; cf.bzee = t1.y; cf.sigma = t1.z; cf.ax = t1.w; cf.ay = t2.x; cf.az = t2.y;
                if (CUBIC) load_cubic(a.table_cubic + (kClassFloats / 4) * cls[t], cf);
            } else {
                cf.bKq = a.coef.bKq; cf.bzee = a.coef.bzee; cf.c4 = a.coef.c4; cf.sigma = a.coef.sigma;
                cf.ax = a.coef.ax; cf.ay = a.coef.ay; cf.az = a.coef.az; cf.mu2 = a.coef.mu2;
                if (CUBIC) { cf.bK1c = a.coef.bK1c; cf.bK2c = a.coef.bK2c; for (int q = 0; q < 9; ++q) cf.cub[q] = a.coef.cub[q]; cf.bK2u = a.coef.bK2u; }
            }
            cf.kx = a.coef.kx * kscale; cf.ky = a.coef.ky * kscale; cf.kz = a.coef.kz * kscale;
            cf.gx = a.coef.gx * kscale; cf.gy = a.coef.gy * kscale;
            float bE = 1.f, bW = 1.f, bN = 1.f, bS = 1.f, bU = HASZ ? 1.f : 0.f, bD = HASZ ? 1.f : 0.f;
            if (MASK || PERCELL) {
                const unsigned b = mb[t];
                bE = (b & 1u) ? 1.f : 0.f;  bW = (b & 2u) ? 1.f : 0.f;
                bN = (b & 4u) ? 1.f : 0.f;  bS = (b & 8u) ? 1.f : 0.f;
                bU = (b & 16u) ? 1.f : 0.f; bD = (b & 32u) ? 1.f : 0.f;
            } else {
                if (nx < 2) { bE = 0.f; bW = 0.f; }
                if (ny < 2) { bN = 0.f; bS = 0.f; }
            }
            float Sg[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float sx = bE * (e[c] - m[c]) + bW * (wv[c] - m[c]);
                const float sy = bN * (N[c] - m[c]) + bS * (S_[c] - m[c]);
                float acc = fmaf(cf.kx, sx, cf.ky * sy);
                if (HASZ) acc = fmaf(cf.kz, bU * (U[c] - m[c]) + bD * (D[c] - m[c]), acc);
                Sg[c] = acc;
            }
            float selfc = 0.5f * fmaf(cf.kx, bE + bW, cf.ky * (bN + bS));
            if (HASZ) selfc = fmaf(0.5f * cf.kz, bU + bD, selfc);
            float dzx = 0.f, dzy = 0.f, dxx = 0.f, dyy = 0.f;
            if (DMI) {
                dzx = bE * e[2] - bW * wv[2];
                dzy = bN * N[2] - bS * S_[2];
                dxx = bE * e[0] - bW * wv[0];
                dyy = bN * N[1] - bS * S_[1];
            }
            const unsigned cell = (unsigned)row * nx + (unsigned)(i0 + 2 * t);       // natural cell index (< 2^31)
            const uint4 rnd = philox4x32_10(make_uint4(cell, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi);
            const CellResult r = cell_update<DMI, false, CUBIC>(m, Sg, selfc, dzx, dzy, dxx, dyy, Bext, Bd, cf, rnd, omc);
            float f0 = m[0], f1 = m[1], f2 = m[2], f3 = r.L;
            if (r.accept) {
                f0 += r.dm[0]; f1 += r.dm[1]; f2 += r.dm[2]; f3 *= r.f;
                a.m[0][ownb + t] = f0; a.m[1][ownb + t] = f1; a.m[2][ownb + t] = f2;
                n_acc++;
            }
            fs0 += f0; fs1 += f1; fs2 += f2; fs3 += f3;
        }
    }
    pass_tail(a, s_tail, n_acc, (act[0] ? 1u : 0u) + (act[1] ? 1u : 0u), fs0, fs1, fs2, fs3, kPass2Threads / 32);
}

// S11 + bookkeeping, one thread: advance the sweep counter; every 100 iterations compare the acceptance rate with
// 0.5 +- 0.05 and move the cone by one degree, clamped to [1, 180] degrees.
__device__ __forceinline__ void end_sweep(Control* ctl)
{
    ctl->sweep += 1ull;
    ctl->run_sweeps += 1ull;
    ctl->win_sweeps += 1u;
    if (ctl->win_sweeps >= 100u) {
        ctl->accepted += ctl->win_accepted; ctl->trials += ctl->win_trials;
        if (ctl->adaptive && ctl->win_trials > 0ull) {
            const double rate = (double)ctl->win_accepted / (double)ctl->win_trials;
            double cone = ctl->cone_deg;
            if (rate > 0.55) cone = fmin(180.0, cone + 1.0);
            else if (rate < 0.45) cone = fmax(1.0, cone - 1.0);
            ctl->cone_deg = cone;
            const double h = sin(0.5 * cone * 0.017453292519943295);
            ctl->one_minus_cos_cone = (float)(2.0 * h * h);
        }
        ctl->win_accepted = 0ull; ctl->win_trials = 0ull; ctl->win_sweeps = 0u;
    }
}
__global__ void end_sweep_kernel(Control* ctl) { end_sweep(ctl); }

// ------------------------------------------------------------------------------------------------ small meshes: all iterations in one launch
// Meshes of a few thousand cells without demag (BASELINE.json config 1: 1024 cells) are bound by launch latency: three
// launches per iteration take ~12 us while the arithmetic of a pass takes ~1 us.  Here ONE CTA runs n iterations in one
// launch (SURVEY 8(d) "Config 1"): red pass, barrier, black pass, barrier, end-of-sweep bookkeeping by thread 0, barrier.
// The cell arithmetic is pass_one_cell, the same function the one-cell pass uses, with coherent loads (a pass reads what
// the previous pass of the same launch wrote; the state lives in this SM's L1/L2); counters and running sums are reduced
// per pass with the same integer arithmetic, so the results are bit-identical to the launch-per-pass path.
constexpr int kSmallThreads = 1024;
constexpr int kSmallMaxCells = 1 << 13;         // <= 4 cells per thread and colour: a warp's fixed-point sum stays inside int32 for |m| < 2

template <unsigned F>
__global__ void __launch_bounds__(kSmallThreads, 1) small_mesh_sweeps_kernel(const SweepArgs a, int n_sweeps)
{
    __shared__ unsigned s_cnt;                        // accepted | trials << 16 would overflow: two words
    __shared__ unsigned s_tri;
    __shared__ long long s_sum[4];
    const int tid = threadIdx.x;
    const int hxr = (a.g.nx + 1) >> 1, rows = a.g.ny * a.g.nz, slots = hxr * rows;
    Control* ctl = a.ctl;
    for (int it = 0; it < n_sweeps; ++it) {
        const unsigned long long sweep = *reinterpret_cast<volatile unsigned long long*>(&ctl->sweep);
        const float omc = *reinterpret_cast<volatile float*>(&ctl->one_minus_cos_cone);
        for (int col = 0; col < 2; ++col) {
            if (tid == 0) { s_cnt = 0u; s_tri = 0u; s_sum[0] = s_sum[1] = s_sum[2] = s_sum[3] = 0; }
            __syncthreads();
            unsigned n_acc = 0u, n_tri = 0u;
            int i0 = 0, i1 = 0, i2 = 0, i3 = 0;       // fixed point per thread: <= 32 cells of |m| < 2 stay inside int32
            for (int idx = tid; idx < slots; idx += kSmallThreads) {
                const int q = idx % hxr, row = idx / hxr, j = row % a.g.ny, k = row / a.g.ny;
                bool active, accept;
                float f0, f1, f2, f3;
                pass_one_cell<F, false, true>(a, col, q, j, k, sweep, omc, active, accept, f0, f1, f2, f3);
                n_acc += accept ? 1u : 0u; n_tri += active ? 1u : 0u;
                i0 += __float2int_rn(f0 * kSumScale); i1 += __float2int_rn(f1 * kSumScale);
                i2 += __float2int_rn(f2 * kSumScale); i3 += __float2int_rn(f3 * kSumScale);
            }
            const unsigned wa = __reduce_add_sync(0xffffffffu, n_acc), wt = __reduce_add_sync(0xffffffffu, n_tri);
            const long long w0 = (long long)__reduce_add_sync(0xffffffffu, i0), w1 = (long long)__reduce_add_sync(0xffffffffu, i1),
                            w2 = (long long)__reduce_add_sync(0xffffffffu, i2), w3 = (long long)__reduce_add_sync(0xffffffffu, i3);
            if ((tid & 31) == 0) {
                atomicAdd(&s_cnt, wa); atomicAdd(&s_tri, wt);
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_sum[0]), (unsigned long long)w0);
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_sum[1]), (unsigned long long)w1);
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_sum[2]), (unsigned long long)w2);
                atomicAdd(reinterpret_cast<unsigned long long*>(&s_sum[3]), (unsigned long long)w3);
            }
            __syncthreads();                          // the pass is complete and visible to the whole CTA
            if (tid == 0) {
                ctl->win_accepted += s_cnt; ctl->win_trials += s_tri;
                if (a.run_sums) for (int t = 0; t < 4; ++t) a.run_sums[t] += (unsigned long long)s_sum[t];
                if (col == 1) end_sweep(ctl);
                __threadfence_block();
            }
        }
        __syncthreads();                              // the new sweep counter and cone are visible
    }
}

int launch_end_sweep(Control* ctl, void* stream)
{
    end_sweep_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(ctl);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// CTA brick 32 x BY x BZ (kPassThreads threads): BZ covers up to 4 layers so that the z neighbours are lines the CTA reads anyway.
static void brick(const Geometry& g, dim3* block, dim3* grid)
{
    const int bz = g.nz >= 4 ? 4 : (g.nz >= 2 ? 2 : 1);
    const int by = kPassThreads / 32 / bz;
    const int hxr = (g.nx + 1) >> 1;
    *block = dim3(32, by, bz);
    *grid = dim3((hxr + 31) / 32, (g.ny + by - 1) / by, (g.nz + bz - 1) / bz);
}

template <unsigned F>
static int launch_variant(const SweepArgs& a, bool debug, cudaStream_t st)
{
    dim3 b, gr; brick(a.g, &b, &gr);
    if (gr.y > 65535u || gr.z > 65535u) return MMC_E_UNSUPPORTED;
    const int hxr = (a.g.nx + 1) >> 1;
#ifndef MMC_PASS_CELLS
#define MMC_PASS_CELLS 2
#endif
    const bool pairable = MMC_PASS_CELLS == 2 && !((a.g.pbc & 1u) && (hxr & 1));        // see colour_pass2_kernel
    if (debug) colour_pass_kernel<F, true><<<gr, b, 0, st>>>(a);
    else if (!pairable) colour_pass_kernel<F, false><<<gr, b, 0, st>>>(a);
    else {
        const int bz = a.g.nz >= 4 ? 4 : (a.g.nz >= 2 ? 2 : 1), by = kPass2Threads / 32 / bz;
        const dim3 b2(32, by, bz), g2((hxr + 63) / 64, (a.g.ny + by - 1) / by, (a.g.nz + bz - 1) / bz);
        if (g2.y > 65535u || g2.z > 65535u) return MMC_E_UNSUPPORTED;
        colour_pass2_kernel<F><<<g2, b2, 0, st>>>(a);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// Instantiated variants: the smallest instantiated superset of the requested features is used.  F_PERCELL must
// match exactly (its word array and table exist only in per-cell mode); the mask and B_d arrays always exist
// (B_d = 0 when the demag term is off), so the other flags may be over-approximated.
// n whole iterations in one launch for small meshes without demag; returns MMC_E_UNSUPPORTED when the mesh does not qualify
// (the caller then takes the launch-per-pass path).  Variants: uniform coefficients only.
int launch_small_mesh_sweeps(const SweepArgs& a, unsigned f, int n_sweeps, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const long long cells = (long long)a.g.nx * a.g.ny * a.g.nz;
    if (cells > kSmallMaxCells || (f & (F_PERCELL | F_DEMAG | F_CUBIC))) return MMC_E_UNSUPPORTED;
    f &= ~F_DENSE;
    constexpr unsigned U = F_MASK | F_Z | F_DMI;
    if (f == 0u) small_mesh_sweeps_kernel<0u><<<1, kSmallThreads, 0, st>>>(a, n_sweeps);
    else if ((f & ~F_MASK) == 0u) small_mesh_sweeps_kernel<F_MASK><<<1, kSmallThreads, 0, st>>>(a, n_sweeps);
    else small_mesh_sweeps_kernel<U><<<1, kSmallThreads, 0, st>>>(a, n_sweeps);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

int launch_colour_pass(const SweepArgs& a, unsigned f, bool debug, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    constexpr unsigned UALL = F_MASK | F_Z | F_DMI | F_DEMAG, PALL = UALL | F_PERCELL;
    const bool dense = (f & F_DENSE) != 0;             // only ever a promise, never over-approximated
    f &= ~F_DENSE;
    if (f & F_CUBIC) {                                 // cubic anisotropy: the all-features variants
        if (f & F_PERCELL) return launch_variant<PALL | F_CUBIC>(a, debug, st);
        return launch_variant<UALL | F_CUBIC>(a, debug, st);
    }
    if (f & F_PERCELL) {
        if (debug) return launch_variant<PALL>(a, true, st);
        if (!(f & F_DMI)) {                                                                                  // cfg 4
            if (dense) return launch_variant<F_MASK | F_PERCELL | F_Z | F_DEMAG | F_DENSE>(a, false, st);
            return launch_variant<F_MASK | F_PERCELL | F_Z | F_DEMAG>(a, false, st);
        }
        return launch_variant<PALL>(a, false, st);
    }
    if (debug) return launch_variant<UALL>(a, true, st);
    if (f == 0u) return launch_variant<0u>(a, false, st);                                                   // cfg 1
    if ((f & ~(F_DEMAG)) == 0u) return launch_variant<F_DEMAG>(a, false, st);
    if ((f & ~(F_MASK | F_DEMAG)) == 0u) {                                                                  // cfg 2 (dense), 5
        if (dense) return launch_variant<F_MASK | F_DEMAG | F_DENSE>(a, false, st);
        return launch_variant<F_MASK | F_DEMAG>(a, false, st);
    }
    if ((f & ~(F_DMI | F_DEMAG)) == 0u) return launch_variant<F_DMI | F_DEMAG>(a, false, st);               // cfg 3
    if ((f & ~(F_MASK | F_Z | F_DEMAG)) == 0u) return launch_variant<F_MASK | F_Z | F_DEMAG>(a, false, st);
    return launch_variant<UALL>(a, false, st);
}

}  // namespace mmc
