// kernels_sweep.cu -- the MMC colour pass (PAPER.md:92 steps 1-4, Eq. (5), (7), (10), (11), (14), (15)) for sm_100a.
//
// One thread owns four consecutive cells of the active colour in one mesh row (one float4 per SoA array of the
// colour-split layout, see mmc_internal.h).  Neighbours are all of the other colour: the y/z neighbours are the
// float4 at the same compact index of the adjacent rows, the x neighbours are the float4 at the same compact
// index of the other colour's row plus one scalar.  All loads are 16-byte, fully coalesced, and every fetched
// sector is used.  RNG: one Philox4x32-10 block per cell per sweep keyed by the natural cell index.
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
        const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}
// 23-bit uniform strictly inside (0,1): ((x>>9) + 0.5) * 2^-23, exact in fp32.
__device__ __forceinline__ float u01(unsigned x) { return fmaf((float)(x >> 9), 1.1920928955078125e-7f, 5.9604644775390625e-8f); }

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float comp(const float4& v, int l) { return l == 0 ? v.x : l == 1 ? v.y : l == 2 ? v.z : v.w; }

struct CellCoef {
    float kx, ky, kz, gx, gy, bKq, bzee, c4, sigma, ax, ay, az;
    double mu2;
};

struct CellResult { float dm[3]; float terms[6]; float margin; bool accept; };

// The per-cell body: trial move (O3), dF/kBT (O4), Eq. (5) in the log domain (O5).
//   m      : current vector          S  : sum_d k_d sum_{bonded nb in d}(m_nb - m)   (beta J_d folded into k_d)
//   selfc  : sum_d k_d n_d / 2       dzx, dzy, dxx, dyy : E-W / N-S differences of m_z, m_x, m_y for the DMI vector
//   B      : B_ext + B_d (tesla) -- or, when SPLIT (debug), Bext and Bd kept apart for the per-term dump
template <bool DMI, bool TERMS>
__device__ __forceinline__ CellResult cell_update(const float m[3], const float S[3], float selfc,
                                                  float dzx, float dzy, float dxx, float dyy,
                                                  const float Bext[3], const float Bd[3],
                                                  const CellCoef& cf, uint4 rnd, float omc)
{
    CellResult r;
    const float u_cos = u01(rnd.x), u_phi = u01(rnd.y), u_len = u01(rnd.z), u_acc = u01(rnd.w);
    const float l2 = fmaf(m[0], m[0], fmaf(m[1], m[1], m[2] * m[2]));
    const float iL = rsqrtf(l2), L = l2 * iL;
    const float n0 = m[0] * iL, n1 = m[1] * iL, n2 = m[2] * iL;
    // tangent frame: a = axis of the smallest |m_a| (raw components, ties -> lowest index); t1 = e_a x n normalised
    const float a0 = fabsf(m[0]), a1 = fabsf(m[1]), a2 = fabsf(m[2]);
    int ax = 0; float amin = a0;
    if (a1 < amin) { ax = 1; amin = a1; }
    if (a2 < amin) { ax = 2; }
    float t10, t11, t12;
    if (ax == 0)      { t10 = 0.f;  t11 = -n2;  t12 = n1; }
    else if (ax == 1) { t10 = n2;   t11 = 0.f;  t12 = -n0; }
    else              { t10 = -n1;  t11 = n0;   t12 = 0.f; }
    const float it = rsqrtf(fmaf(t10, t10, fmaf(t11, t11, t12 * t12)));
    t10 *= it; t11 *= it; t12 *= it;
    const float t20 = n1 * t12 - n2 * t11, t21 = n2 * t10 - n0 * t12, t22 = n0 * t11 - n1 * t10;   // n x t1
    const float w = u_cos * omc;                       // 1 - cos(theta), uniform on the cap
    const float st = sqrtf(w * (2.f - w));
    float sp, cp;
    sincospif(2.f * u_phi, &sp, &cp);
    const float ca = st * cp, sa = st * sp;
    const float dn0 = fmaf(ca, t10, fmaf(sa, t20, -w * n0));
    const float dn1 = fmaf(ca, t11, fmaf(sa, t21, -w * n1));
    const float dn2 = fmaf(ca, t12, fmaf(sa, t22, -w * n2));
    const float s = cf.sigma * fmaf(2.f, u_len, -1.f);  // f = 1 + s
    const float f = 1.f + s;
    const float dm0 = L * fmaf(f, dn0, s * n0), dm1 = L * fmaf(f, dn1, s * n1), dm2 = L * fmaf(f, dn2, s * n2);
    r.dm[0] = dm0; r.dm[1] = dm1; r.dm[2] = dm2;
    // exchange: -dm.S + selfc |dm|^2
    const float dmsq = fmaf(dm0, dm0, fmaf(dm1, dm1, dm2 * dm2));
    const float ex = fmaf(selfc, dmsq, -fmaf(dm0, S[0], fmaf(dm1, S[1], dm2 * S[2])));
    // uniaxial anisotropy: -beta V Kq (dm.e)((2m+dm).e)
    const float dme = fmaf(dm0, cf.ax, fmaf(dm1, cf.ay, dm2 * cf.az));
    const float sme = fmaf(fmaf(2.f, m[0], dm0), cf.ax, fmaf(fmaf(2.f, m[1], dm1), cf.ay, fmaf(2.f, m[2], dm2) * cf.az));
    const float an = -cf.bKq * dme * sme;
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
    // longitudinal: dl2 c4 (2 (l2 - mu2) + dl2), dl2 = |m'|^2 - |m|^2 = l2 s (2 + s); the bracket l2 - mu2 cancels
    // 2-3 digits below Tc, so it is formed in fp64 from the exact squares of the stored fp32 components
    const double l2d = fma((double)m[0], (double)m[0], fma((double)m[1], (double)m[1], (double)m[2] * (double)m[2]));
    const float dev = (float)(l2d - cf.mu2);
    const float dl2 = l2 * (s * (2.f + s));
    const float lng = dl2 * cf.c4 * fmaf(2.f, dev, dl2);
    const float dF = ((ex + an) + (zee + dem)) + (dmi + lng);
    // Eq. (5): accept iff ln u < 4 ln f - dF
    r.margin = __logf(u_acc) - 4.f * __logf(f) + dF;
    r.accept = r.margin < 0.f;
    if (TERMS) { r.terms[0] = ex; r.terms[1] = an; r.terms[2] = zee; r.terms[3] = dmi; r.terms[4] = dem; r.terms[5] = lng; }
    return r;
}

// ------------------------------------------------------------------------------------------------ the pass
template <unsigned F, bool DEBUG>
__global__ void __launch_bounds__(256) colour_pass_kernel(const SweepArgs a, const int rows_first)
{
    constexpr bool MASK = (F & F_MASK) != 0, PERCELL = (F & F_PERCELL) != 0, HASZ = (F & F_Z) != 0,
                   DMI = (F & F_DMI) != 0, DEMAG = (F & F_DEMAG) != 0;
    const Geometry g = a.g;
    const int cpr = g.hx >> 2;                       // float4 chunks per row
    const int R = g.ny * g.nz;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int chunk, rr;
    if (rows_first) {                                // consecutive warps walk rows at one 128-cell x block
        const long long gw = tid >> 5;
        const int xb = (int)(gw / R);
        rr = (int)(gw - (long long)xb * R);
        chunk = xb * 32 + (threadIdx.x & 31);
    } else {
        rr = (int)(tid / cpr);
        chunk = (int)(tid - (long long)rr * cpr);
    }
    const bool in_range = rr < R && chunk < cpr;
    int acc_cnt = 0, tri_cnt = 0;
    float sum0 = 0.f, sum1 = 0.f, sum2 = 0.f, sum3 = 0.f;

    if (in_range) {
        int j, k;
        if (HASZ) { j = rr / g.nz; k = rr - j * g.nz; } else { j = rr; k = 0; }
        const int col = a.colour;
        const int s = ((j + k) & 1) ^ col;           // active cells of this row sit at i = 2q + s
        const int q0 = chunk << 2;
        const int row = k * g.ny + j;
        const int hxr = (g.nx + 1) >> 1;             // compact length of the real (unpadded) row
        const long long ownb = (long long)col * g.H + (long long)row * g.hx + q0;
        const long long othc = (long long)(1 - col) * g.H;
        const long long othb = othc + (long long)row * g.hx + q0;
        // neighbour rows (wrap when periodic, else clamp: an out-of-mesh neighbour is never bonded)
        int jn = j + 1, js = j - 1;
        if (jn == g.ny) jn = (g.pbc & 2u) ? 0 : j;
        if (js < 0) js = (g.pbc & 2u) ? g.ny - 1 : j;
        const long long nb_n = othc + (long long)(k * g.ny + jn) * g.hx + q0;
        const long long nb_s = othc + (long long)(k * g.ny + js) * g.hx + q0;
        long long nb_u = 0, nb_d = 0;
        if (HASZ) {
            int ku = k + 1, kd = k - 1;
            if (ku == g.nz) ku = (g.pbc & 4u) ? 0 : k;
            if (kd < 0) kd = (g.pbc & 4u) ? g.nz - 1 : k;
            nb_u = othc + (long long)(ku * g.ny + j) * g.hx + q0;
            nb_d = othc + (long long)(kd * g.ny + j) * g.hx + q0;
        }
        // the one x neighbour outside this thread's float4 of the other colour
        int qe = (s == 0) ? q0 - 1 : q0 + 4;
        if (qe < 0) qe = (g.pbc & 1u) ? hxr - 1 : 0;
        if (qe >= hxr) qe = (g.pbc & 1u) ? 0 : q0;
        const long long exb = othc + (long long)row * g.hx + qe;

        float4 own[3], ox[3], yn[3], ys[3], zu[3], zd[3], bd[3];
        float oe[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            own[c] = ld4(a.m[c] + ownb);
            ox[c] = ldg4(a.m[c] + othb);
            yn[c] = ldg4(a.m[c] + nb_n);
            ys[c] = ldg4(a.m[c] + nb_s);
            oe[c] = __ldg(a.m[c] + exb);
            if (HASZ) { zu[c] = ldg4(a.m[c] + nb_u); zd[c] = ldg4(a.m[c] + nb_d); }
            if (DEMAG) bd[c] = ldg4(a.bd[c] + ownb);
        }
        unsigned mask4 = 0x7f7f7f7fu;
        if (MASK) mask4 = __ldg(reinterpret_cast<const unsigned*>(a.mask + ownb));
        float4 p_invT, p_c4, p_mh, p_ml, p_bKq, p_bzee, p_sig, p_ax, p_ay, p_az;
        if (PERCELL) {
            p_invT = ldg4(a.pc.invT + ownb); p_c4 = ldg4(a.pc.c4 + ownb);
            p_mh = ldg4(a.pc.mu2hi + ownb);  p_ml = ldg4(a.pc.mu2lo + ownb);
            p_bKq = ldg4(a.pc.bKq + ownb);   p_bzee = ldg4(a.pc.bzee + ownb);
            p_sig = ldg4(a.pc.sigma + ownb);
            p_ax = ldg4(a.pc.ax + ownb); p_ay = ldg4(a.pc.ay + ownb); p_az = ldg4(a.pc.az + ownb);
        }
        const unsigned long long sweep = a.ctl->sweep;
        const float omc = a.ctl->one_minus_cos_cone;
        const float Bext[3] = { a.coef.Bx, a.coef.By, a.coef.Bz };
        const long long nat_row = (long long)row * g.nx;
        float outm[3][4];
        bool any_acc = false;

#pragma unroll
        for (int l = 0; l < 4; ++l) {
            const unsigned mb = (mask4 >> (8 * l)) & 0xffu;
            const float m[3] = { comp(own[0], l), comp(own[1], l), comp(own[2], l) };
            outm[0][l] = m[0]; outm[1][l] = m[1]; outm[2][l] = m[2];
            if (MASK && !(mb & 0x40u)) continue;                         // empty or padding slot
            const int q = q0 + l;
            const int i = 2 * q + s;
            // x neighbours (E = i+1, W = i-1) of the other colour
            float e[3], wv[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float in4_same = comp(ox[c], l);
                if (s == 0) { e[c] = in4_same; wv[c] = (l == 0) ? oe[c] : comp(ox[c], l - 1); }
                else        { wv[c] = in4_same; e[c] = (l == 3) ? oe[c] : comp(ox[c], l + 1); }
            }
            if (MASK && s == 1 && l < 3 && q == hxr - 1 && (g.pbc & 1u)) {   // ragged periodic row: E wraps to q = 0
#pragma unroll
                for (int c = 0; c < 3; ++c) e[c] = __ldg(a.m[c] + othc + (long long)row * g.hx);
            }
            CellCoef cf;
            float kscale = 1.f;
            if (PERCELL) {
                kscale = comp(p_invT, l);
                cf.bKq = comp(p_bKq, l); cf.bzee = comp(p_bzee, l); cf.c4 = comp(p_c4, l); cf.sigma = comp(p_sig, l);
                cf.ax = comp(p_ax, l); cf.ay = comp(p_ay, l); cf.az = comp(p_az, l);
                cf.mu2 = (double)comp(p_mh, l) + (double)comp(p_ml, l);
            } else {
                cf.bKq = a.coef.bKq; cf.bzee = a.coef.bzee; cf.c4 = a.coef.c4; cf.sigma = a.coef.sigma;
                cf.ax = a.coef.ax; cf.ay = a.coef.ay; cf.az = a.coef.az; cf.mu2 = a.coef.mu2;
            }
            cf.kx = a.coef.kx * kscale; cf.ky = a.coef.ky * kscale; cf.kz = a.coef.kz * kscale;
            cf.gx = a.coef.gx * kscale; cf.gy = a.coef.gy * kscale;
            // bond weights (1 or 0)
            float bE = 1.f, bW = 1.f, bN = 1.f, bS = 1.f, bU = HASZ ? 1.f : 0.f, bD = HASZ ? 1.f : 0.f;
            if (MASK) {
                bE = (mb & 1u) ? 1.f : 0.f;  bW = (mb & 2u) ? 1.f : 0.f;
                bN = (mb & 4u) ? 1.f : 0.f;  bS = (mb & 8u) ? 1.f : 0.f;
                bU = (mb & 16u) ? 1.f : 0.f; bD = (mb & 32u) ? 1.f : 0.f;
            } else {
                if (g.nx < 2) { bE = 0.f; bW = 0.f; }
                if (g.ny < 2) { bN = 0.f; bS = 0.f; }
            }
            float S[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float sx = bE * (e[c] - m[c]) + bW * (wv[c] - m[c]);
                const float sy = bN * (comp(yn[c], l) - m[c]) + bS * (comp(ys[c], l) - m[c]);
                float acc = fmaf(cf.kx, sx, cf.ky * sy);
                if (HASZ) acc = fmaf(cf.kz, bU * (comp(zu[c], l) - m[c]) + bD * (comp(zd[c], l) - m[c]), acc);
                S[c] = acc;
            }
            float selfc = 0.5f * fmaf(cf.kx, bE + bW, cf.ky * (bN + bS));
            if (HASZ) selfc = fmaf(0.5f * cf.kz, bU + bD, selfc);
            float dzx = 0.f, dzy = 0.f, dxx = 0.f, dyy = 0.f;
            if (DMI) {
                dzx = bE * e[2] - bW * wv[2];
                dzy = bN * comp(yn[2], l) - bS * comp(ys[2], l);
                dxx = bE * e[0] - bW * wv[0];
                dyy = bN * comp(yn[1], l) - bS * comp(ys[1], l);
            }
            float Bd[3] = { 0.f, 0.f, 0.f };
            if (DEMAG) { Bd[0] = comp(bd[0], l); Bd[1] = comp(bd[1], l); Bd[2] = comp(bd[2], l); }
            const unsigned long long cell = (unsigned long long)(nat_row + i);
            const uint4 rnd = philox4x32_10(make_uint4((unsigned)cell, (unsigned)(cell >> 32), (unsigned)sweep, (unsigned)(sweep >> 32)),
                                            a.seed_lo, a.seed_hi);
            const CellResult r = cell_update<DMI, DEBUG>(m, S, selfc, dzx, dzy, dxx, dyy, Bext, Bd, cf, rnd, omc);
            tri_cnt++;
            if (r.accept) {
                acc_cnt++; any_acc = true;
                outm[0][l] = m[0] + r.dm[0]; outm[1][l] = m[1] + r.dm[1]; outm[2][l] = m[2] + r.dm[2];
            }
            sum0 += outm[0][l]; sum1 += outm[1][l]; sum2 += outm[2][l];
            sum3 += sqrtf(fmaf(outm[0][l], outm[0][l], fmaf(outm[1][l], outm[1][l], outm[2][l] * outm[2][l])));
            if (DEBUG) {
                const long long c = (long long)cell;
                if (a.dbg_dm) { a.dbg_dm[3 * c] = r.dm[0]; a.dbg_dm[3 * c + 1] = r.dm[1]; a.dbg_dm[3 * c + 2] = r.dm[2]; }
                if (a.dbg_terms) for (int t = 0; t < 6; ++t) a.dbg_terms[6 * c + t] = r.terms[t];
                if (a.dbg_margin) a.dbg_margin[c] = r.margin;
                if (a.dbg_acc) a.dbg_acc[c] = r.accept ? 1 : 0;
            }
        }
        if (any_acc) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
                *reinterpret_cast<float4*>(a.m[c] + ownb) = make_float4(outm[c][0], outm[c][1], outm[c][2], outm[c][3]);
        }
    }

    // ---- S10: acceptance counters (exact integers) and running sums of the final vectors, per block
    __shared__ int s_cnt[8][2];
    __shared__ float s_sum[8][4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc_cnt += __shfl_xor_sync(0xffffffffu, acc_cnt, o);
        tri_cnt += __shfl_xor_sync(0xffffffffu, tri_cnt, o);
        sum0 += __shfl_xor_sync(0xffffffffu, sum0, o);
        sum1 += __shfl_xor_sync(0xffffffffu, sum1, o);
        sum2 += __shfl_xor_sync(0xffffffffu, sum2, o);
        sum3 += __shfl_xor_sync(0xffffffffu, sum3, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
        s_cnt[warp][0] = acc_cnt; s_cnt[warp][1] = tri_cnt;
        s_sum[warp][0] = sum0; s_sum[warp][1] = sum1; s_sum[warp][2] = sum2; s_sum[warp][3] = sum3;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int ac = 0, tc = 0; double d0 = 0, d1 = 0, d2 = 0, d3 = 0;
        const int nw = blockDim.x >> 5;
        for (int w = 0; w < nw; ++w) {
            ac += s_cnt[w][0]; tc += s_cnt[w][1];
            d0 += s_sum[w][0]; d1 += s_sum[w][1]; d2 += s_sum[w][2]; d3 += s_sum[w][3];
        }
        if (tc) {
            atomicAdd(&a.ctl->win_trials, (unsigned long long)tc);
            if (ac) atomicAdd(&a.ctl->win_accepted, (unsigned long long)ac);
        }
        if (a.run_sums) {                            // one slot per block: fixed summation order, no fp atomics
            double* slot = a.run_sums + 4ll * blockIdx.x;
            slot[0] += d0; slot[1] += d1; slot[2] += d2; slot[3] += d3;
        }
    }
}

// S11 + bookkeeping, one thread: advance the sweep counter; every 100 iterations compare the acceptance rate with
// 0.5 +- 0.05 and move the cone by one degree, clamped to [1, 180] degrees.
__global__ void end_sweep_kernel(Control* ctl)
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

int launch_end_sweep(Control* ctl, double*, int, void* stream)
{
    end_sweep_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(ctl);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

int sweep_grid_blocks(const Geometry& g, bool)
{
    const long long cpr = g.hx >> 2, R = (long long)g.ny * g.nz;
    long long threads;
    if (cpr >= 32 && cpr % 32 == 0) threads = cpr * R;
    else threads = cpr * R;
    return (int)((threads + 255) / 256);
}

template <unsigned F>
static int launch_variant(const SweepArgs& a, bool debug, cudaStream_t st)
{
    const long long cpr = a.g.hx >> 2;
    const int rows_first = (cpr >= 32 && cpr % 32 == 0) ? 1 : 0;
    const int blocks = sweep_grid_blocks(a.g, true);
    if (debug) colour_pass_kernel<F, true><<<blocks, 256, 0, st>>>(a, rows_first);
    else       colour_pass_kernel<F, false><<<blocks, 256, 0, st>>>(a, rows_first);
    return cudaGetLastError() == cudaSuccess ? MMC_OK : MMC_E_CUDA;
}

// Instantiated variants: the smallest instantiated superset of the requested features is used.  F_PERCELL must
// match exactly (its arrays exist only in per-cell mode); the mask and B_d arrays always exist (B_d = 0 when the
// demag term is off), so the other flags may be over-approximated.
int launch_colour_pass(const SweepArgs& a, unsigned f, bool, bool debug, void* stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    constexpr unsigned UALL = F_MASK | F_Z | F_DMI | F_DEMAG, PALL = UALL | F_PERCELL;
    if (f & F_PERCELL) {
        if (debug) return launch_variant<PALL>(a, true, st);
        if (!(f & F_DMI)) return launch_variant<F_MASK | F_PERCELL | F_Z | F_DEMAG>(a, false, st);          // cfg 4
        return launch_variant<PALL>(a, false, st);
    }
    if (debug) return launch_variant<UALL>(a, true, st);
    if (f == 0u) return launch_variant<0u>(a, false, st);                                                   // cfg 1
    if ((f & ~(F_DEMAG)) == 0u) return launch_variant<F_DEMAG>(a, false, st);
    if ((f & ~(F_MASK | F_DEMAG)) == 0u) return launch_variant<F_MASK | F_DEMAG>(a, false, st);             // cfg 2, 5
    if ((f & ~(F_DMI | F_DEMAG)) == 0u) return launch_variant<F_DMI | F_DEMAG>(a, false, st);               // cfg 3
    if ((f & ~(F_MASK | F_Z | F_DEMAG)) == 0u) return launch_variant<F_MASK | F_Z | F_DEMAG>(a, false, st);
    return launch_variant<UALL>(a, false, st);
}

}  // namespace mmc
