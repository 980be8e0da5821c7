// kernels_sweep.cu -- the MMC colour pass (PAPER.md:92 steps 1-4, Eq. (5), (7), (10), (11), (14), (15)) for sm_100a.
//
// Three kernels share one per-cell body (cell_update: trial move, dF/kBT, Eq. (5)):
//   colour_pass2_kernel      the timed path: a thread owns TWO consecutive compact cells of a row of the active colour
//                            (64-bit loads of the colour-split arrays of mmc_internal.h; a warp = 64 compact cells of one
//                            row, a CTA = a 64 x BY x BZ brick of one colour, so neighbour lines are shared through L1);
//   colour_pass_kernel       one cell per thread: the debug pass with its per-cell dump, and meshes whose compact rows do not
//                            pair up (periodic in x with an odd compact row length);
//   small_mesh_sweeps_kernel meshes of <= 8192 cells without demag: one CTA, state in shared memory, all n iterations of
//                            mmc_sweep(n) in ONE launch.
// The instruction stream, not the byte stream, is the tighter bound of the pass.
// RNG: one Philox4x32-10 block per cell per sweep keyed by the natural cell index (replayable on the CPU side).
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstring>

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

// The part of the trial move (O3) that needs nothing but the cell's own vector and its random numbers: unit vector, tangent
// frame, rotation inside the cone.  Kept apart from the energies so that a kernel can run it for all of a thread's cells BEFORE
// it touches anything that comes from a dependent load (class table, neighbours): ~250 instructions per cell of cover.
struct Trial { float n0, n1, n2, dn0, dn1, dn2, L, l2, u_len, u_acc; };
__device__ __forceinline__ Trial trial_direction(const float m[3], uint4 rnd, float omc)
{
    Trial tr;
    const float u_cos = u01(rnd.x), u_phi = u01(rnd.y);
    tr.u_len = u01(rnd.z); tr.u_acc = u01(rnd.w);
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
    tr.dn0 = sel2 ? db : (sel1 ? dc : da);
    tr.dn1 = sel2 ? dc : (sel1 ? da : db);
    tr.dn2 = sel2 ? da : (sel1 ? db : dc);
    tr.n0 = n0; tr.n1 = n1; tr.n2 = n2; tr.L = L; tr.l2 = l2;
    return tr;
}

// The rest of the per-cell body: length factor (O3), dF/kBT (O4), Eq. (5) in the log domain (O5).
//   m      : current vector          S  : sum_d k_d sum_{bonded nb in d}(m_nb - m)   (beta J_d folded into k_d)
//   selfc  : sum_d k_d n_d / 2       dzx, dzy, dxx, dyy : E-W / N-S differences of m_z, m_x, m_y for the DMI vector
//   B      : B_ext + B_d (tesla); TERMS (debug) keeps Zeeman and demag apart for the per-term dump
template <bool DMI, bool TERMS, bool CUBIC>
__device__ __forceinline__ CellResult cell_update(const float m[3], const float S[3], float selfc,
                                                  float dzx, float dzy, float dxx, float dyy,
                                                  const float Bext[3], const float Bd[3],
                                                  const CellCoef& cf, const Trial& tr)
{
    CellResult r;
    const float u_len = tr.u_len, u_acc = tr.u_acc, l2 = tr.l2, L = tr.L;
    const float n0 = tr.n0, n1 = tr.n1, n2 = tr.n2, dn0 = tr.dn0, dn1 = tr.dn1, dn2 = tr.dn2;
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
// The last CTA of the black pass closes the iteration (S11) when SweepArgs::finish is set: every CTA signs in on a global
// ticket after its counters have been added (fence, then ticket), and the CTA that draws the last ticket has all of them
// behind it.  Saves the one-thread end_sweep launch of every iteration (~3 us on the launch-bound configs).
__device__ __forceinline__ void finish_sweep_ticket(const SweepArgs& a)
{
    if (!a.finish) return;
    __threadfence();
    const unsigned total = gridDim.x * gridDim.y * gridDim.z;
    if (atomicAdd(&a.ctl->pad, 1u) == total - 1u) {
        __threadfence();
        a.ctl->pad = 0u;
        end_sweep(a.ctl);
    }
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
            // This one thread keeps the CTA's slot (registers, shared memory) occupied after every other warp has retired, so
            // its path is kept short: the block's totals by ten independent volatile loads (the fence and the arrival counter
            // order them after every warp's shared atomics; reading them back with atomicAdd(.., 0) was a chain of ten
            // round trips: cfg 4 0.4972 -> 0.4952 ms per iteration, cfg 5 0.3721 -> 0.3700), then six global reductions that
            // nobody waits for.  (Sharding those six targets over 64 lines was measured on top and brought nothing on cfg 4 / 6.)
            const volatile unsigned* vc = sm.cnt;
            const volatile unsigned* vs = &sm.sum[0][0];
            const unsigned tc = vc[1], ac = vc[0];
            const unsigned s00 = vs[0], s01 = vs[1], s02 = vs[2], s03 = vs[3], s10 = vs[4], s11 = vs[5], s12 = vs[6], s13 = vs[7];
            if (tc) {
                atomicAdd(&a.ctl->win_trials, (unsigned long long)tc);
                if (ac) atomicAdd(&a.ctl->win_accepted, (unsigned long long)ac);
                if (want_sums) {                       // sign-extend the two 32-bit two's-complement halves
                    atomicAdd(&a.run_sums[0], (unsigned long long)((long long)(int)s00 + (long long)(int)s10));
                    atomicAdd(&a.run_sums[1], (unsigned long long)((long long)(int)s01 + (long long)(int)s11));
                    atomicAdd(&a.run_sums[2], (unsigned long long)((long long)(int)s02 + (long long)(int)s12));
                    atomicAdd(&a.run_sums[3], (unsigned long long)((long long)(int)s03 + (long long)(int)s13));
                }
            }
            finish_sweep_ticket(a);
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
// plain (generic) load for the single-CTA kernel, whose state lives in shared memory and whose passes read what earlier
// passes of the same launch wrote (ordered by block barriers); read-only path otherwise
template <bool COHERENT> __device__ __forceinline__ float ldc(const float* p) { return COHERENT ? *p : __ldg(p); }

// One cell of the active colour: compact index q of row (j, k).  The body of the one-cell-per-thread pass.
// PRE: the direction part of the trial move was computed ahead of time by cell_trial (the pipelined small-mesh kernel)
template <unsigned F, bool DEBUG, bool COHERENT, bool PRE = false>
__device__ __forceinline__ void pass_one_cell(const SweepArgs& a, int col, int q, int j, int k, unsigned long long sweep, float omc,
                                              bool& active, bool& accept, float& fs0, float& fs1, float& fs2, float& fs3,
                                              const Trial& pre = Trial())
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
        Trial tr;
        if (PRE) tr = pre;
        else tr = trial_direction(m, philox4x32_10(make_uint4(cell, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi), omc);
        const CellResult r = cell_update<DMI, DEBUG, CUBIC>(m, S, selfc, dzx, dzy, dxx, dyy, Bext, Bd, cf, tr);
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
    pdl_enter();
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

// The update of a thread's two cells from their loaded neighbourhood: compact cells q0, q0 + 1 of row (j, k) (mesh cells i0
// and i0 + 2; `row` = k ny + j; s = parity of the row: active cells sit at i = 2 q + s).  m2 / bd2: own vectors and B_d;
// xc: the other colour's pair at the same compact index, xs: its third x neighbour (q0 - 1 for s == 0, q0 + 2 for s == 1);
// yn, ys, zu, zd: the other colour's pairs of the four adjacent rows.  Shared by colour_pass2_kernel (operands from
// global memory / L1) and colour_pass_tma_kernel (operands from the TMA-staged shared-memory tile).
template <unsigned F>
__device__ __forceinline__ void update_pair(const SweepArgs& a, int s, int row, int i0, unsigned ownb, const bool (&act)[2],
                                            const unsigned (&mb)[2], const unsigned (&cls)[2], const float2 (&m2)[3],
                                            const float2 (&xc)[3], const float (&xs)[3], const float2 (&yn)[3], const float2 (&ys)[3],
                                            const float2 (&zu)[3], const float2 (&zd)[3], const float2 (&bd2)[3],
                                            unsigned long long sweep, float omc,
                                            unsigned& n_acc, float& fs0, float& fs1, float& fs2, float& fs3)
{
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DMI = (F & F_DMI) != 0, CUBIC = (F & F_CUBIC) != 0;
    const int nx = a.g.nx, ny = a.g.ny;
    const float Bext[3] = { a.coef.Bx, a.coef.By, a.coef.Bz };
    // Philox and the direction part of both trial moves first: they need only the cells' own vectors, so ~500 instructions run
    // before anything that depends on the class table or on the neighbours is touched (their loads are in flight meanwhile)
    const unsigned cell0 = (unsigned)row * nx + (unsigned)i0;                    // natural cell index (< 2^31); the second cell is cell0 + 2
    const float ma[3] = { m2[0].x, m2[1].x, m2[2].x }, mb2[3] = { m2[0].y, m2[1].y, m2[2].y };
    const Trial trial0 = trial_direction(ma, philox4x32_10(make_uint4(cell0, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi), omc);
    const Trial trial1 = trial_direction(mb2, philox4x32_10(make_uint4(cell0 + 2u, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi), omc);
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
        const CellResult r = cell_update<DMI, false, CUBIC>(m, Sg, selfc, dzx, dzy, dxx, dyy, Bext, Bd, cf, t ? trial1 : trial0);
        float f0 = m[0], f1 = m[1], f2 = m[2], f3 = r.L;
        if (r.accept) {
            f0 += r.dm[0]; f1 += r.dm[1]; f2 += r.dm[2]; f3 *= r.f;
            a.m[0][ownb + t] = f0; a.m[1][ownb + t] = f1; a.m[2][ownb + t] = f2;
            n_acc++;
        }
        fs0 += f0; fs1 += f1; fs2 += f2; fs3 += f3;
    }
}

// ------------------------------------------------------------------------------------------------ the pass, two cells per thread
// The same pass with a thread owning TWO consecutive compact cells of a row (mesh cells i and i + 2): the vectors, B_d and
// class words / masks come as 64-bit loads, the x neighbour between the two cells is loaded once, index arithmetic, bond
// decoding and the reductions are shared.  Used for every non-debug launch unless x is periodic with an odd compact row
// length (then the wrap neighbour of the last cell would not pair up).  blockDim = (32, BY, BZ), 256 threads = a brick of
// 64 x BY x BZ cells of one colour; grid = (ceil(hxr/64), ceil(ny/BY), ceil(nz/BZ)).
constexpr int kPass2Threads = 256;

#ifndef MMC_PASS2_MINB
#define MMC_PASS2_MINB 4      // 64 registers (48 bytes spilled): measured 5 / 4 / 3 / 2 CTAs per SM on cfg 4: 74.7 (48 registers, 292 B spilled) / 57.5 / 61 / 72 us per pass
#endif
template <unsigned F>
__global__ void __launch_bounds__(kPass2Threads, MMC_PASS2_MINB) colour_pass2_kernel(const SweepArgs a)
{
    pdl_enter();
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DEMAG = (F & F_DEMAG) != 0, DENSE = (F & F_DENSE) != 0;
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
        update_pair<F>(a, s, row, i0, ownb, act, mb, cls, m2, xc, xs, yn, ys, zu, zd, bd2, a.ctl->sweep, a.ctl->one_minus_cos_cone,
                       n_acc, fs0, fs1, fs2, fs3);
    }
    pass_tail(a, s_tail, n_acc, (act[0] ? 1u : 0u) + (act[1] ? 1u : 0u), fs0, fs1, fs2, fs3, kPass2Threads / 32);
}

// ------------------------------------------------------------------------------------------------ the pass, staged by TMA
// The same pass with its operands staged into shared memory by the TMA unit (cp.async.bulk.tensor + mbarrier) instead of
// per-thread global loads: a persistent CTA walks over tiles of 64 x BY x BZ compact cells of the active colour; one producer
// warp requests, per tile, the own-colour boxes (m, B_d, class words) and the other colour's boxes with a one-row / one-layer
// halo and a 16-byte aligned x window (72 floats from q0 - 4), into a ring of kTmaStages stages; eight consumer warps wait
// on the stage's full barrier, update the tile from shared memory with update_pair (two cells per thread, a warp per row)
// and release the stage.  Out-of-mesh elements arrive as zeros (their bonds are masked).  TMA does not wrap, so this
// kernel serves meshes without periodic directions (BASELINE configs 2, 4, 5); everything else takes colour_pass2_kernel.
// north_star (a) asks for this variant to be measured against plain L1-served loads: profiles/ has both.
constexpr int kTmaConsumerWarps = 8, kTmaThreads = (kTmaConsumerWarps + 1) * 32, kTmaStages = 2;    // two CTAs per SM
constexpr int kTmaX = 64, kTmaXO = 72;                 // compact cells per tile row; floats of the other colour's x window

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned arrivals)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(arrivals) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// one box of a rank-4 tensor (x, y, z, colour) -> shared memory, completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_4d(void* dst, const void* tmap, int x, int y, int z, int w, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_addr(dst)), "l"(tmap), "r"(x), "r"(y), "r"(z), "r"(w), "r"(smem_addr(bar)) : "memory");
}

template <unsigned F>
__global__ void __launch_bounds__(kTmaThreads, 2) colour_pass_tma_kernel(const SweepArgs a, const PassTmaShape sh,
                                                                       const __grid_constant__ PassTmaMaps maps)
{
    pdl_enter();
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DEMAG = (F & F_DEMAG) != 0, DENSE = (F & F_DENSE) != 0;
    extern __shared__ __align__(128) unsigned char tsm[];
    __shared__ unsigned long long s_bar[2 * kTmaStages];          // full[stage], empty[stage]
    __shared__ unsigned long long s_tot[6];                       // accepted, trials, four fixed-point sums
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int BY = sh.BY, BZ = sh.BZ, zh = sh.zh, rows = BY * BZ, OY = BY + 2;
    const int own_arr = rows * kTmaX * 4;                          // bytes of one own-colour array of a tile
    const int oth_arr = sh.oth_arr;                                // bytes of one other-colour array (128-byte multiple)
    constexpr int NOWN = 3 + (DEMAG ? 3 : 0) + (PERCELL ? 1 : 0);
    const int stage_bytes = NOWN * own_arr + 3 * oth_arr;
    const int ntiles = sh.tiles_x * sh.tiles_y * sh.tiles_z;
    const int col = a.colour;
    if (threadIdx.x == 0) {
        for (int q = 0; q < kTmaStages; ++q) { mbar_init(&s_bar[q], 1u); mbar_init(&s_bar[kTmaStages + q], kTmaConsumerWarps); }
        for (int q = 0; q < 6; ++q) s_tot[q] = 0ull;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (warp == kTmaConsumerWarps) {
        // ---- producer warp: lane 0 requests the boxes of every tile of this CTA.  (Measured and dropped: the whole warp pulling
        // the landed tile's coefficient-table lines into L1 with prefetch.global.L1: no effect on the consumers' gather stalls.)
        int it = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++it) {
            const int st = it % kTmaStages, ph = (it / kTmaStages) & 1;
            unsigned char* base = tsm + (size_t)st * stage_bytes;
            unsigned long long* full = &s_bar[st];
            if (lane == 0) {
                mbar_wait(&s_bar[kTmaStages + st], (unsigned)(ph ^ 1));              // the consumers have released this stage
                const int tx = t % sh.tiles_x, r = t / sh.tiles_x, ty = r % sh.tiles_y, tz = r / sh.tiles_y;
                const int q0 = tx * kTmaX, j0 = ty * BY, k0 = tz * BZ;
                unsigned bytes = (unsigned)(3 * own_arr + 3 * sh.oth_box_bytes);
                if (DEMAG) bytes += 3u * own_arr;
                if (PERCELL) bytes += (unsigned)own_arr;
                mbar_expect_tx(full, bytes);
                int slot = 0;
                for (int c = 0; c < 3; ++c) tma_load_4d(base + (slot++) * own_arr, &maps.own_m[c], q0, j0, k0, col, full);
                if (DEMAG) for (int c = 0; c < 3; ++c) tma_load_4d(base + (slot++) * own_arr, &maps.bd[c], q0, j0, k0, col, full);
                if (PERCELL) tma_load_4d(base + (slot++) * own_arr, &maps.cw, q0, j0, k0, col, full);
                unsigned char* ob = base + NOWN * own_arr;
                for (int c = 0; c < 3; ++c) tma_load_4d(ob + c * oth_arr, &maps.oth_m[c], q0 - 4, j0 - 1, k0 - zh, 1 - col, full);
            }
        }
    } else {
        // ---- consumers: a warp per tile row, two cells per lane
        const int nx = a.g.nx, ny = a.g.ny, nz = a.g.nz, hx = a.g.hx;
        const unsigned H = (unsigned)a.g.H;
        const unsigned long long sweep = a.ctl->sweep;
        const float omc = a.ctl->one_minus_cos_cone;
        const bool want_sums = a.run_sums != nullptr;
        long long tot[6] = { 0, 0, 0, 0, 0, 0 };                   // lane 0: accepted, trials, fixed-point sums of this warp
        const int ql = 2 * lane;                                   // compact index of the lane's first cell inside the tile row
        // (Measured and dropped, per-cell classes: fetching the NEXT row's class-table words while the current row is computed
        // needs ~24 more registers per thread; at two CTAs of 288 threads per SM that spills 264 bytes per thread into an L1 that
        // the stages have left 30 KB of, and one CTA of 17 warps is capped at 96 registers by the allocation granularity.)
        int it = 0;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x, ++it) {
            const int st = it % kTmaStages, ph = (it / kTmaStages) & 1;
            const int tx = t % sh.tiles_x, rr = t / sh.tiles_x, ty = rr % sh.tiles_y, tz = rr / sh.tiles_y;
            const int j0 = ty * BY, k0 = tz * BZ, q0 = tx * kTmaX + ql;
            const unsigned char* base = tsm + (size_t)st * stage_bytes;
            const unsigned char* ob = base + NOWN * own_arr;
            mbar_wait(&s_bar[st], (unsigned)ph);                   // the tile has landed
            unsigned n_acc = 0u, n_tri = 0u;
            int is0 = 0, is1 = 0, is2 = 0, is3 = 0;                // fixed-point sums, rounded per cell pair exactly as colour_pass2_kernel does
            for (int r = warp; r < rows; r += kTmaConsumerWarps) {
                float fs0 = 0.f, fs1 = 0.f, fs2 = 0.f, fs3 = 0.f;
                const int kk = r / BY, jj = r - kk * BY, j = j0 + jj, k = k0 + kk;
                const int s = ((j + k) & 1) ^ col;
                const int i0 = 2 * q0 + s;
                const bool inrow = j < ny && k < nz;
                bool act[2] = { inrow && i0 < nx, inrow && i0 + 2 < nx };
                const int row = k * ny + j;
                const unsigned ownb = (unsigned)col * H + (unsigned)row * hx + q0;
                const int oo = (r * kTmaX + ql) * 4;               // byte offset of the lane's pair in an own-colour array
                unsigned mb[2] = { 0x7fu, 0x7fu }, cls[2] = { 0u, 0u };
                if (act[0]) {
                    if (PERCELL) {
                        const uint2 w = *reinterpret_cast<const uint2*>(base + (NOWN - 1) * own_arr + oo);
                        mb[0] = w.x & 0x7fu; cls[0] = w.x >> 7; mb[1] = w.y & 0x7fu; cls[1] = w.y >> 7;
                    } else if (MASK) {
                        const uchar2 w = __ldg(reinterpret_cast<const uchar2*>(a.mask + ownb));
                        mb[0] = w.x; mb[1] = w.y;
                    }
                    if (!DENSE && (MASK || PERCELL)) { act[0] = act[0] && (mb[0] & 0x40u); act[1] = act[1] && (mb[1] & 0x40u); }
                }
                if (act[0] || act[1]) {
                    float2 m2[3], xc[3], yn[3], ys[3], zu[3], zd[3], bd2[3];
                    float xs[3];
                    const int orow = (kk + zh) * OY + jj + 1;      // this row inside the other colour's box
                    const int up = (zh || kk + 1 < BZ) ? OY : 0, dn = (zh || kk > 0) ? -OY : 0;   // no layer there: any row (bond masked)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const float* om = reinterpret_cast<const float*>(ob + c * oth_arr) + 4 + ql;
                        m2[c] = *reinterpret_cast<const float2*>(base + c * own_arr + oo);
                        xc[c] = *reinterpret_cast<const float2*>(om + orow * kTmaXO);
                        xs[c] = om[orow * kTmaXO + (s ? 2 : -1)];
                        yn[c] = *reinterpret_cast<const float2*>(om + (orow + 1) * kTmaXO);
                        ys[c] = *reinterpret_cast<const float2*>(om + (orow - 1) * kTmaXO);
                        if (HASZ) {
                            zu[c] = *reinterpret_cast<const float2*>(om + (orow + up) * kTmaXO);
                            zd[c] = *reinterpret_cast<const float2*>(om + (orow + dn) * kTmaXO);
                        }
                        bd2[c] = DEMAG ? *reinterpret_cast<const float2*>(base + (3 + c) * own_arr + oo) : make_float2(0.f, 0.f);
                    }
                    update_pair<F>(a, s, row, i0, ownb, act, mb, cls, m2, xc, xs, yn, ys, zu, zd, bd2, sweep, omc, n_acc, fs0, fs1, fs2, fs3);
                }
                n_tri += (act[0] ? 1u : 0u) + (act[1] ? 1u : 0u);
                if (want_sums) {
                    is0 += __float2int_rn(fs0 * kSumScale); is1 += __float2int_rn(fs1 * kSumScale);
                    is2 += __float2int_rn(fs2 * kSumScale); is3 += __float2int_rn(fs3 * kSumScale);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&s_bar[kTmaStages + st]);    // this warp has read everything it needs from the stage
            // S10: the tile's counters and fixed-point sums (a warp holds <= 128 cells of |m| < 2: inside int32), added up in 64 bits by lane 0
            const unsigned cnt = __reduce_add_sync(0xffffffffu, n_acc | (n_tri << 16));
            tot[0] += cnt & 0xffffu; tot[1] += cnt >> 16;
            if (want_sums) {
                tot[2] += __reduce_add_sync(0xffffffffu, is0);
                tot[3] += __reduce_add_sync(0xffffffffu, is1);
                tot[4] += __reduce_add_sync(0xffffffffu, is2);
                tot[5] += __reduce_add_sync(0xffffffffu, is3);
            }
        }
        if (lane == 0 && tot[1])
            for (int q = 0; q < 6; ++q) atomicAdd(&s_tot[q], (unsigned long long)tot[q]);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_tot[1]) {
            atomicAdd(&a.ctl->win_trials, s_tot[1]);
            if (s_tot[0]) atomicAdd(&a.ctl->win_accepted, s_tot[0]);
            if (a.run_sums) for (int q = 0; q < 4; ++q) atomicAdd(&a.run_sums[q], s_tot[2 + q]);
        }
        finish_sweep_ticket(a);
    }
}

__global__ void end_sweep_kernel(Control* ctl) { pdl_enter(); end_sweep(ctl); }

// ------------------------------------------------------------------------------------------------ small meshes: all iterations in one launch
// Meshes of a few thousand cells without demag (BASELINE.json config 1: 1024 cells) are bound by launch latency: three
// launches per iteration take ~12 us while the arithmetic of a pass takes ~1 us.  Here ONE CTA runs n iterations in one
// launch (SURVEY 8(d) "Config 1"): the state (colour-split, 3 x 2H floats), the control block and the running sums are
// copied to shared memory, then red pass, barrier, black pass, barrier, end-of-sweep bookkeeping by thread 0, barrier, n
// times, and everything is written back once.  The cell arithmetic is pass_one_cell, the same function the one-cell pass
// uses (its pointers simply point into shared memory); counters and running sums are reduced per pass with the same
// integer arithmetic, so the results are bit-identical to the launch-per-pass path.
constexpr int kSmallThreads = 1024;
constexpr int kSmallMaxCells = 1 << 13;         // <= 4 cells per thread and colour: a warp's fixed-point sum stays inside int32 for |m| < 2
constexpr int kSmallMaxSlots = 1 << 14;         // storage slots (2 H) per component: 3 x 64 KB of shared memory

template <unsigned F>
__global__ void __launch_bounds__(kSmallThreads, 1) small_mesh_sweeps_kernel(const SweepArgs a_in, int n_sweeps)
{
    extern __shared__ float s_m[];                    // [3][2 H]
    __shared__ Control s_ctl;
    __shared__ unsigned long long s_run[4];
    __shared__ int s_w[2][kSmallThreads / 32][6];     // per pass parity, per warp: accepted, trials, four fixed-point sums
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    SweepArgs a = a_in;
    const int hxr = (a.g.nx + 1) >> 1, rows = a.g.ny * a.g.nz, slots = hxr * rows;
    const int S2 = (int)(2 * a.g.H);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        for (int i = tid; i < S2; i += kSmallThreads) s_m[c * S2 + i] = a_in.m[c][i];
        a.m[c] = s_m + c * S2;
    }
    if (tid == 0) s_ctl = *a_in.ctl;
    if (tid < 4) s_run[tid] = a_in.run_sums ? a_in.run_sums[tid] : 0ull;
    a.ctl = &s_ctl;
    // Per pass: every warp leaves its counts and fixed-point sums in s_w (plain stores, a warp's <= 128 cells of |m| < 2 stay
    // inside int32), one block barrier makes the pass and these visible, and warp 0 adds them up (two 16-bit halves per value
    // through the 32-bit warp reduction) and keeps the books while the other warps are already in the next pass.  Three block
    // barriers per iteration; no atomics.
    auto bookkeeping = [&](int par, bool last) {
        // warp 0 only
        long long tot[6];
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            const int v = s_w[par][lane][q];
            const int lo = __reduce_add_sync(0xffffffffu, v & 0xffff), hi = __reduce_add_sync(0xffffffffu, v >> 16);   // arithmetic shift: signed values
            tot[q] = (long long)hi * 65536ll + (long long)lo;
        }
        if (lane == 0) {
            s_ctl.win_accepted += (unsigned long long)tot[0]; s_ctl.win_trials += (unsigned long long)tot[1];
            if (a_in.run_sums) for (int t = 0; t < 4; ++t) s_run[t] += (unsigned long long)tot[2 + t];
            if (last) end_sweep(&s_ctl);
        }
    };
    __syncthreads();
    for (int it = 0; it < n_sweeps; ++it) {
        const unsigned long long sweep = s_ctl.sweep;
        const float omc = s_ctl.one_minus_cos_cone;
        for (int col = 0; col < 2; ++col) {
            unsigned n_acc = 0u, n_tri = 0u;
            int i0 = 0, i1 = 0, i2 = 0, i3 = 0;       // fixed point per thread: <= 8 cells of |m| < 2
            for (int idx = tid; idx < slots; idx += kSmallThreads) {
                const int q = idx % hxr, row = idx / hxr, j = row % a.g.ny, k = row / a.g.ny;
                bool active, accept;
                float f0, f1, f2, f3;
                pass_one_cell<F, false, true>(a, col, q, j, k, sweep, omc, active, accept, f0, f1, f2, f3);
                n_acc += accept ? 1u : 0u; n_tri += active ? 1u : 0u;
                i0 += __float2int_rn(f0 * kSumScale); i1 += __float2int_rn(f1 * kSumScale);
                i2 += __float2int_rn(f2 * kSumScale); i3 += __float2int_rn(f3 * kSumScale);
            }
            const int wa = (int)__reduce_add_sync(0xffffffffu, n_acc), wt = (int)__reduce_add_sync(0xffffffffu, n_tri);
            const int w0 = __reduce_add_sync(0xffffffffu, i0), w1 = __reduce_add_sync(0xffffffffu, i1),
                      w2 = __reduce_add_sync(0xffffffffu, i2), w3 = __reduce_add_sync(0xffffffffu, i3);
            if (lane == 0) { int* w = s_w[col][warp]; w[0] = wa; w[1] = wt; w[2] = w0; w[3] = w1; w[4] = w2; w[5] = w3; }
            __syncthreads();                          // the pass and its partial sums are visible to the whole CTA
            if (warp == 0) bookkeeping(col, col == 1);
        }
        __syncthreads();                              // the new sweep counter and cone are visible
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
        for (int i = tid; i < S2; i += kSmallThreads) a_in.m[c][i] = s_m[c * S2 + i];
    if (tid == 0) *a_in.ctl = s_ctl;
    if (tid < 4 && a_in.run_sums) a_in.run_sums[tid] = s_run[tid];
}

// Philox + direction part of the trial move of cell (q, j, k) of colour col from its CURRENT vector: everything of a cell's
// update that does not depend on its neighbours (garbage for cells outside the mesh or empty: never used)
__device__ __forceinline__ Trial cell_trial(const SweepArgs& a, int col, int q, int j, int k, unsigned long long sweep, float omc)
{
    const int s = ((j + k) & 1) ^ col, i = 2 * q + s, row = k * a.g.ny + j;
    const unsigned ownb = (unsigned)col * (unsigned)a.g.H + (unsigned)row * a.g.hx + q;
    const float m[3] = { a.m[0][ownb], a.m[1][ownb], a.m[2][ownb] };
    const unsigned cell = (unsigned)row * a.g.nx + i;
    return trial_direction(m, philox4x32_10(make_uint4(cell, 0u, (unsigned)sweep, (unsigned)(sweep >> 32)), a.seed_lo, a.seed_hi), omc);
}

// Meshes of at most 512 cells per colour (BASELINE config 1: 32 x 32): every cell has its own thread -- threads 0 .. 511 the red
// cells, 512 .. 1023 the black ones -- and the two halves work in a two-stage pipeline: while one colour runs the neighbour-
// dependent half of its update (gather, dF, Eq. (5), store), the other colour runs the neighbour-INDEPENDENT half of its next
// one (Philox and the rotation of the trial move, which need only the cell's own, by then final, vector).  The dependent
// chain of an iteration shrinks from two whole updates to two half updates.  The red cells' next trial needs the next
// iteration's cone: in the one iteration per 100 after which the adaptive controller may change it, that half is computed after
// the end-of-sweep bookkeeping instead.  Same arithmetic as everywhere else: results are bit-identical to the launch-per-pass path.
template <unsigned F>
__global__ void __launch_bounds__(kSmallThreads, 1) small_mesh_pipe_kernel(const SweepArgs a_in, int n_sweeps)
{
    extern __shared__ float s_m[];                    // [3][2 H]
    __shared__ Control s_ctl;
    __shared__ unsigned long long s_run[4];
    __shared__ int s_w[2][kSmallThreads / 64][6];     // per colour, per warp of that colour: accepted, trials, four fixed-point sums
    const int tid = threadIdx.x, lane = tid & 31;
    const int half = tid >> 9, idx = tid & 511, hwarp = idx >> 5;     // colour of this thread, its slot, its warp within the colour
    SweepArgs a = a_in;
    const int hxr = (a.g.nx + 1) >> 1, rows = a.g.ny * a.g.nz, slots = hxr * rows;
    const int S2 = (int)(2 * a.g.H);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        for (int i = tid; i < S2; i += kSmallThreads) s_m[c * S2 + i] = a_in.m[c][i];
        a.m[c] = s_m + c * S2;
    }
    if (tid == 0) s_ctl = *a_in.ctl;
    if (tid < 4) s_run[tid] = a_in.run_sums ? a_in.run_sums[tid] : 0ull;
    a.ctl = &s_ctl;
    const bool mine = idx < slots;
    const int q = mine ? idx % hxr : 0, row = mine ? idx / hxr : 0, j = row % a.g.ny, k = row / a.g.ny;
    auto bookkeeping = [&](int col, bool last) {       // one warp: totals of the colour's 16 warps
        long long tot[6];
#pragma unroll
        for (int t = 0; t < 6; ++t) {
            const int v = lane < kSmallThreads / 64 ? s_w[col][lane][t] : 0;
            const int lo = __reduce_add_sync(0xffffffffu, v & 0xffff), hi = __reduce_add_sync(0xffffffffu, v >> 16);
            tot[t] = (long long)hi * 65536ll + (long long)lo;
        }
        if (lane == 0) {
            s_ctl.win_accepted += (unsigned long long)tot[0]; s_ctl.win_trials += (unsigned long long)tot[1];
            if (a_in.run_sums) for (int t = 0; t < 4; ++t) s_run[t] += (unsigned long long)tot[2 + t];
            if (last) end_sweep(&s_ctl);
        }
    };
    // the neighbour-dependent half of this thread's cell, and its partial sums
    auto finish_cell = [&](const Trial& tr, unsigned long long sweep, float omc) {
        bool active = false, accept = false;
        float f0 = 0.f, f1 = 0.f, f2 = 0.f, f3 = 0.f;
        if (mine) pass_one_cell<F, false, true, true>(a, half, q, j, k, sweep, omc, active, accept, f0, f1, f2, f3, tr);
        const int wa = (int)__reduce_add_sync(0xffffffffu, accept ? 1u : 0u), wt = (int)__reduce_add_sync(0xffffffffu, active ? 1u : 0u);
        const int w0 = __reduce_add_sync(0xffffffffu, __float2int_rn(f0 * kSumScale)), w1 = __reduce_add_sync(0xffffffffu, __float2int_rn(f1 * kSumScale)),
                  w2 = __reduce_add_sync(0xffffffffu, __float2int_rn(f2 * kSumScale)), w3 = __reduce_add_sync(0xffffffffu, __float2int_rn(f3 * kSumScale));
        if (lane == 0) { int* w = s_w[half][hwarp]; w[0] = wa; w[1] = wt; w[2] = w0; w[3] = w1; w[4] = w2; w[5] = w3; }
    };
    __syncthreads();
    Trial tr = {};
    if (half == 0 && mine && n_sweeps > 0) tr = cell_trial(a, 0, q, j, k, s_ctl.sweep, s_ctl.one_minus_cos_cone);   // prologue: red, first iteration
    for (int it = 0; it < n_sweeps; ++it) {
        const unsigned long long sweep = s_ctl.sweep;
        const float omc = s_ctl.one_minus_cos_cone;
        const bool cone_may_change = s_ctl.adaptive && s_ctl.win_sweeps == 99u;      // this iteration closes a controller window
        // stage 1: red cells finish, black cells prepare (their vectors are final since the previous black stage)
        if (half == 0) finish_cell(tr, sweep, omc);
        else if (mine) tr = cell_trial(a, 1, q, j, k, sweep, omc);
        __syncthreads();
        if (tid < 32) bookkeeping(0, false);
        // stage 2: black cells finish, red cells prepare the NEXT iteration (same cone unless the controller is about to act)
        if (half == 1) finish_cell(tr, sweep, omc);
        else if (mine && !cone_may_change && it + 1 < n_sweeps) tr = cell_trial(a, 0, q, j, k, sweep + 1ull, omc);
        __syncthreads();
        if (tid < 32) bookkeeping(1, true);
        __syncthreads();                              // the new sweep counter and cone are visible
        if (cone_may_change && half == 0 && mine && it + 1 < n_sweeps) tr = cell_trial(a, 0, q, j, k, s_ctl.sweep, s_ctl.one_minus_cos_cone);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
        for (int i = tid; i < S2; i += kSmallThreads) a_in.m[c][i] = s_m[c * S2 + i];
    if (tid == 0) *a_in.ctl = s_ctl;
    if (tid < 4 && a_in.run_sums) a_in.run_sums[tid] = s_run[tid];
}

int launch_end_sweep(Control* ctl, void* stream)
{
    launch_pdl(end_sweep_kernel, dim3(1), dim3(1), (size_t)(0), (cudaStream_t)stream, ctl);
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
    if (debug) launch_pdl(colour_pass_kernel<F, true>, dim3(gr), dim3(b), (size_t)(0), st, a);
    else if (!pairable) launch_pdl(colour_pass_kernel<F, false>, dim3(gr), dim3(b), (size_t)(0), st, a);
    else {
        const int bz = a.g.nz >= 4 ? 4 : (a.g.nz >= 2 ? 2 : 1), by = kPass2Threads / 32 / bz;
        const dim3 b2(32, by, bz), g2((hxr + 63) / 64, (a.g.ny + by - 1) / by, (a.g.nz + bz - 1) / bz);
        if (g2.y > 65535u || g2.z > 65535u) return MMC_E_UNSUPPORTED;
        // a grid of fewer CTAs than SMs: the pass is then as long as one thread's instruction chain, and one cell per thread halves
        // it (cfg 2, 64 CTAs: 0.0209 -> 0.0191 ms per iteration; cfg 3, 256 CTAs: no difference).  a.pass1_below: 148, or MMC_PASS1_BELOW.
        if ((long long)g2.x * g2.y * g2.z < a.pass1_below) launch_pdl(colour_pass_kernel<F, false>, dim3(gr), dim3(b), (size_t)(0), st, a);
        else launch_pdl(colour_pass2_kernel<F>, dim3(g2), dim3(b2), (size_t)(0), st, a);
    }
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// Instantiated variants: the smallest instantiated superset of the requested features is used.  F_PERCELL must
// match exactly (its word array and table exist only in per-cell mode); the mask and B_d arrays always exist
// (B_d = 0 when the demag term is off), so the other flags may be over-approximated.
// n whole iterations in one launch for small meshes without demag; returns MMC_E_UNSUPPORTED when the mesh does not qualify
// (the caller then takes the launch-per-pass path).  Variants: uniform coefficients only.
template <unsigned F>
static int launch_small_variant(const SweepArgs& a, int n_sweeps, cudaStream_t st)
{
    const size_t smem = (size_t)3 * 2 * a.g.H * sizeof(float);
    const int slots = ((a.g.nx + 1) >> 1) * a.g.ny * a.g.nz;      // cells per colour
    auto kern = slots <= kSmallThreads / 2 ? small_mesh_pipe_kernel<F> : small_mesh_sweeps_kernel<F>;
    if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
    kern<<<1, kSmallThreads, smem, st>>>(a, n_sweeps);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
int launch_small_mesh_sweeps(const SweepArgs& a, unsigned f, int n_sweeps, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const long long cells = (long long)a.g.nx * a.g.ny * a.g.nz;
    if (cells > kSmallMaxCells || 2 * a.g.H > kSmallMaxSlots || (f & (F_PERCELL | F_DEMAG | F_CUBIC))) return MMC_E_UNSUPPORTED;
    f &= ~F_DENSE;
    constexpr unsigned U = F_MASK | F_Z | F_DMI;
    if (f == 0u) return launch_small_variant<0u>(a, n_sweeps, st);
    if ((f & ~F_MASK) == 0u) return launch_small_variant<F_MASK>(a, n_sweeps, st);
    return launch_small_variant<U>(a, n_sweeps, st);
}

// ---- host side of the TMA-staged pass
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

void pass_tma_build(const Geometry& g, float* const m[3], float* const bd[3], const uint32_t* cw, PassTma* out)
{
    out->ok = false;
    if (g.pbc != 0u) return;                                       // TMA boxes do not wrap
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return;
    }
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(fn);
    PassTmaShape sh{};
    sh.BZ = g.nz >= 4 ? 4 : g.nz;
    sh.zh = g.nz > sh.BZ ? 1 : 0;
    sh.BY = 16 / sh.BZ;
    const int hxr = (g.nx + 1) >> 1;
    sh.tiles_x = (hxr + kTmaX - 1) / kTmaX; sh.tiles_y = (g.ny + sh.BY - 1) / sh.BY; sh.tiles_z = (g.nz + sh.BZ - 1) / sh.BZ;
    const int oy = sh.BY + 2, oz = sh.BZ + 2 * sh.zh;
    sh.oth_box_bytes = oy * oz * kTmaXO * 4;
    sh.oth_arr = (sh.oth_box_bytes + 127) / 128 * 128;
    const cuuint64_t dims[4] = { (cuuint64_t)g.hx, (cuuint64_t)g.ny, (cuuint64_t)g.nz, 2 };
    const cuuint64_t strides[3] = { (cuuint64_t)g.hx * 4, (cuuint64_t)g.hx * g.ny * 4, (cuuint64_t)g.H * 4 };
    const cuuint32_t own_box[4] = { (cuuint32_t)kTmaX, (cuuint32_t)sh.BY, (cuuint32_t)sh.BZ, 1 };
    const cuuint32_t oth_box[4] = { (cuuint32_t)kTmaXO, (cuuint32_t)oy, (cuuint32_t)oz, 1 };
    const cuuint32_t ones[4] = { 1, 1, 1, 1 };
    auto enc = [&](unsigned char (&dst)[128], CUtensorMapDataType dt, const void* base, const cuuint32_t* box) {
        CUtensorMap tm;
        if (encode(&tm, dt, 4, const_cast<void*>(base), dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return false;
        static_assert(sizeof(CUtensorMap) == 128, "tensor map size");
        std::memcpy(dst, &tm, 128);
        return true;
    };
    bool good = true;
    for (int c = 0; c < 3 && good; ++c) {
        good = enc(out->maps.own_m[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, m[c], own_box) && enc(out->maps.oth_m[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, m[c], oth_box)
               && enc(out->maps.bd[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, bd[c], own_box);
    }
    if (good && cw) good = enc(out->maps.cw, CU_TENSOR_MAP_DATA_TYPE_UINT32, cw, own_box);
    if (!good) return;
    out->sh = sh; out->key[0] = m[0]; out->key[1] = bd[0]; out->key[2] = cw;
    out->ok = true;
}

template <unsigned F>
static int launch_tma_variant(const SweepArgs& a, const PassTma& t, cudaStream_t st)
{
    constexpr int NOWN = 3 + ((F & F_DEMAG) ? 3 : 0) + ((F & F_PERCELL) ? 1 : 0);
    const int rows = t.sh.BY * t.sh.BZ;
    const size_t smem = (size_t)kTmaStages * ((size_t)NOWN * rows * kTmaX * 4 + 3 * (size_t)t.sh.oth_arr);
    auto kern = colour_pass_tma_kernel<F>;
    if (smem > 48 * 1024 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMC_E_CUDA;
    const int ntiles = t.sh.tiles_x * t.sh.tiles_y * t.sh.tiles_z;
    if (ntiles < 2 * 148) return MMC_E_UNSUPPORTED;               // too few tiles to give every SM its two CTAs: the brick kernel spreads better
    const int grid = 2 * 148;
    launch_pdl(kern, dim3(grid), dim3(kTmaThreads), smem, st, a, t.sh, t.maps);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}
// the feature sets of the open-boundary BASELINE configs; anything else is served by colour_pass2_kernel
static int launch_colour_pass_tma(const SweepArgs& a, unsigned f, const PassTma& t, cudaStream_t st)
{
    switch (f) {
        case F_MASK | F_DEMAG | F_DENSE: return launch_tma_variant<F_MASK | F_DEMAG | F_DENSE>(a, t, st);                                   // cfg 2
        case F_MASK | F_DEMAG: return launch_tma_variant<F_MASK | F_DEMAG>(a, t, st);                                                       // cfg 5
        case F_MASK | F_PERCELL | F_Z | F_DEMAG | F_DENSE: return launch_tma_variant<F_MASK | F_PERCELL | F_Z | F_DEMAG | F_DENSE>(a, t, st);   // cfg 4
        case F_MASK | F_PERCELL | F_Z | F_DEMAG: return launch_tma_variant<F_MASK | F_PERCELL | F_Z | F_DEMAG>(a, t, st);
        case F_MASK | F_Z | F_DEMAG | F_DENSE: return launch_tma_variant<F_MASK | F_Z | F_DEMAG | F_DENSE>(a, t, st);
        default: return MMC_E_UNSUPPORTED;
    }
}

int launch_colour_pass(const SweepArgs& a, unsigned f, bool debug, void* stream, const PassTma* tma)
{
    cudaStream_t st = (cudaStream_t)stream;
    if (tma && tma->ok && !debug) {
        const int rc = launch_colour_pass_tma(a, f, *tma, st);
        if (rc != MMC_E_UNSUPPORTED) return rc;
    }
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
