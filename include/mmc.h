/*
 * mmc.h -- C ABI of the B200-native micromagnetic Monte Carlo (MMC) hot path of
 * arXiv:2106.05593 (S. Lepadatu, "Micromagnetic Monte Carlo method with variable magnetization
 * length based on the LLB equation").  Citations are /root/reference/PAPER.md line numbers.
 *
 * What the library computes: n MMC iterations on a cuboidal mesh of cells of volume
 * V = dx*dy*dz.  One iteration = [demagnetising field by zero-padded FFT convolution
 * with the Newell tensor, Eq. (14), frozen for the iteration] -> red colour pass
 * -> black colour pass (checkerboard).  In a colour pass every non-empty cell of that
 * colour gets exactly one compound trial move (rotation inside a cone + length factor in
 * [1-sigma, 1+sigma], PAPER.md:92 steps 1-2), scored by the local free-energy change
 * (exchange Eq. (10), uniaxial anisotropy Eq. (11), applied field, interfacial DMI Eq. (15),
 * demag Eq. (14), longitudinal term = exponent of Eq. (7)) and accepted with Eq. (5).
 * Random numbers: Philox4x32-10, key = seed, counter = (cell index, sweep counter); one block of
 * four uniforms per cell per sweep, so an oracle can replay the identical stream.
 *
 * Conventions
 *  - every function returns 0 (MMC_OK) or a negative MMC_E_* code; nothing throws or aborts across
 *    the ABI; mmc_last_error(ctx) gives a message for the last failing call on that ctx.
 *  - cell index c = i + nx*(j + ny*k), x fastest; colour = (i+j+k) & 1 (0 = "red").
 *  - m = M/Ms0, stored as three fp32 arrays; all arithmetic of the sweep is fp32
 *    except the longitudinal bracket (fp64).  Fields in tesla, energies in joule.
 *  - pointers documented "device" are plain device pointers valid on the ctx device (for example
 *    torch.Tensor.data_ptr()); "host" pointers are ordinary host memory.  The caller owns every
 *    buffer it passes; the library copies host inputs during the call and keeps no caller pointer.
 *  - all device work is enqueued on the stream given at mmc_create; setters taking host arrays and
 *    mmc_get_observables synchronise that stream, everything else is asynchronous.
 *  - a ctx is not thread-safe; there is no global state.
 */
#ifndef MMC_H_
#define MMC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MMC_OK              0
#define MMC_E_INVALID      -1   /* bad argument (NULL, non-positive size, T <= 0, odd periodic length, ...) */
#define MMC_E_ZERO_LENGTH  -2   /* a non-empty cell has |m| = 0: rotation undefined, length move cannot leave 0 */
#define MMC_E_CUDA         -3   /* a CUDA runtime / cuFFT call failed; see mmc_last_error */
#define MMC_E_NOMEM        -4   /* host or device allocation failed */
#define MMC_E_UNSUPPORTED  -5   /* valid request outside what is built (e.g. A0 differing between regions) */
#define MMC_E_STATE        -6   /* call order: m / material / temperature not set before sweeping */
#define MMC_E_TOO_LARGE    -7   /* mmc_mean_m_static: more cells than its fixed device scratch array serves */

typedef struct mmc_ctx mmc_ctx;   /* opaque, owned by the library */

/* Material of one region, SI units.  Ms0 == 0 marks an empty region (no trial, no bond, no demag source).
 * A0: exchange stiffness at T=0 (A(T) = A0 me^2); K1 + unit axis (ax,ay,az): uniaxial
 * anisotropy constant at T=0 (K1(T) = K1 me^3, Eq. (11)); D0: interfacial DMI at T=0
 * (D(T) = D0 me^2, Eq. (15)); Tc: Curie temperature; mu_atom: atomic moment in J/T
 * (Eq. (8)).  A0 and D0 must be equal in all non-empty regions (MMC_E_UNSUPPORTED).
 * Cubic anisotropy, Eq. (12): K1c, K2c = 4th / 6th order constants at T = 0 in J/m^3,
 * F = V K1c(T) [a^2 b^2 + a^2 g^2 + b^2 g^2] + V K2c(T) a^2 b^2 g^2 with a, b, g the direction cosines of m with respect
 * to the cubic axes and K(T) = K me^(l(l+1)/2), l = 4 and 6; zero at and above Tc.  (c1x,c1y,c1z) and
 * (c2x,c2y,c2z) give two of the axes (orthonormalised by Gram-Schmidt; the third is their cross product); they are
 * ignored when K1c = K2c = 0 and must not be parallel otherwise. */
typedef struct {
    double Ms0, A0, K1, ax, ay, az, D0, Tc, mu_atom;
    double K1c, K2c, c1x, c1y, c1z, c2x, c2y, c2z;
    double K2;      /* 4th-order uniaxial constant of Eq. (11) at T = 0, J/m^3, same axis as K1: F = V K2(T) [1 - (m.e)^2/me^2]^2, K2(T) = K2 me^10 */
} mmc_material;

/* Read-out (PAPER.md:100 acceptance rate; PAPER.md:135 average magnetisation; Appendix B energies).
 * Means are over non-empty cells.  Energies in joule with pair terms counted once:
 * E_ex = sum_bonds (A0 V/h^2)|m_i-m_j|^2, E_an = sum V[K1(T) - K1 me (m.e)^2] + the cubic energy of Eq. (12), E_zee = -V sum Ms0 m.B_ext,
 * E_dmi = -D0 V sum m.G, E_demag = -(V/2) sum Ms0 m.B_d (B_d of the current state), E_long = sum kB T F_l. */
typedef struct {
    double   mean_m[3], mean_len;
    double   E_ex, E_an, E_zee, E_dmi, E_demag, E_long;
    uint64_t accepted, trials, sweeps_done;      /* accepted/trials since creation or the last counter reset */
    double   cone_deg, sigma_used;               /* sigma_used: the (first non-empty cell's) length half-width */
    double   run_mean_m[3], run_mean_len;        /* average of the per-sweep means since mmc_reset_averages */
    uint64_t run_sweeps;
} mmc_obs;

/* Create a context for an nx*ny*nz mesh of dx*dy*dz metre cells on CUDA device `device`.
 * pbc_mask bit0/1/2 = periodic in x/y/z for exchange and DMI (a periodic length must be even and >= 2:
 * the checkerboard needs it); the demag convolution is always open-boundary.  cuda_stream is a
 * cudaStream_t (NULL = legacy default stream).  Defaults: one non-magnetic region, T unset, B = 0,
 * cone 30 deg fixed, sigma from Eq. (13), demag off, seed 0, sweep counter 0. */
int mmc_create(mmc_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz,
               unsigned pbc_mask, int device, void* cuda_stream);
int mmc_destroy(mmc_ctx* ctx);

/* regions: host array of n_regions records; region_of_cell: host int32[N] (NULL => every cell region 0). */
int mmc_set_material(mmc_ctx* ctx, int n_regions, const mmc_material* regions, const int32_t* region_of_cell);
/* 0 => bonds between cells of different regions carry no exchange and no DMI ("phase separation"). */
int mmc_set_exchange_coupling(mmc_ctx* ctx, int inter_region_exchange);
/* Uniform temperature, or per cell when T_per_cell (host float[N], kelvin) is not NULL.
 * Recomputes me (Eq. (9), H_ext = 0), chi (Eq. (8)), the longitudinal coefficients (Eq. (7)) and sigma (Eq. (13)). */
int mmc_set_temperature(mmc_ctx* ctx, double T_uniform, const float* T_per_cell);
int mmc_set_field(mmc_ctx* ctx, double Bx, double By, double Bz);                 /* applied field, tesla */
/* cone half-angle in degrees (0 < cone <= 180); sigma < 0 => Eq. (13) capped at 0.03, else the
 * given half-width of the uniform length factor; adaptive_cone != 0 => every 100 iterations the cone changes by
 * 1 degree when the acceptance rate leaves 0.5 +- 0.05, clamped to [1, 180]. */
int mmc_set_move(mmc_ctx* ctx, double cone_deg, double sigma, int adaptive_cone);
/* updates_per_sweep: 1 = once per iteration; 2 = also before the black pass. */
int mmc_set_demag(mmc_ctx* ctx, int enabled, int updates_per_sweep);
int mmc_set_seed(mmc_ctx* ctx, uint64_t seed);
int mmc_set_sweep_counter(mmc_ctx* ctx, uint64_t sweep);
/* device pointers, N floats each, natural cell order.  m = M/Ms0.  Fails with MMC_E_ZERO_LENGTH if a non-empty
 * cell is 0 or not finite (reading G13) and with MMC_E_INVALID if a non-empty cell has |m| >= 2 (the running sums of the
 * pass are exact fixed-point numbers for |m| < 2; |m| ~ 1000 means M in A/m was passed).  Values in EMPTY cells are
 * ignored, whatever they are (NaN markers included): the library stores 0 there and mmc_get_m returns 0 for them.
 * The check runs when material and temperature are known (here, or at the first call that needs the state). */
int mmc_set_m(mmc_ctx* ctx, const float* mx, const float* my, const float* mz);
int mmc_get_m(mmc_ctx* ctx, float* mx, float* my, float* mz);
/* The same with HOST pointers (N floats each; pinned memory makes the copies asynchronous): the library does the
 * host<->device copies on the ctx stream.  mmc_set_m_host returns after the zero-length check (synchronises);
 * mmc_get_m_host only enqueues: the buffers are valid after the next synchronising call (mmc_get_observables) or a
 * stream synchronise by the caller.  This is the end-to-end path of a caller whose state lives on the host. */
int mmc_set_m_host(mmc_ctx* ctx, const float* mx, const float* my, const float* mz);
int mmc_get_m_host(mmc_ctx* ctx, float* mx, float* my, float* mz);
/* n iterations, asynchronous on the ctx stream.  Launch structure (results do not depend on it, bit for bit):
 * meshes of <= 8192 cells without demag run all n iterations in ONE launch of a single-CTA kernel (state in shared memory);
 * otherwise the first iteration after a change of settings is enqueued kernel by kernel and the rest are replayed from CUDA
 * graphs of 16 and 1 iterations (rebuilt when a setter changes a kernel argument).  Environment knobs, read when the ctx (or
 * its demag plan) is created, for A/B measurements: MMC_NO_GRAPH (plain launches), MMC_PDL=1 (programmatic dependent launch
 * between the kernels of an iteration: measured slower, off by default), MMC_TMA=1 (TMA-staged colour pass on meshes
 * without periodic directions), MMC_LP=1 (layer-pair columns kernel of the demag convolution on multi-layer meshes), MMC_COLS8=1
 * (multi-layer meshes, padded ny 1024 .. 4096: columns kernel with eight instead of sixteen points per thread; measured slower),
 * MMC_DEMAG_GENERIC=1 (the any-length
 * shared-memory FFT kernels of the convolution also where the register-resident ones apply: 2 - 3 times slower, for tests),
 * MMC_PASS1_BELOW=<n> (colour passes whose grid has fewer than n CTAs run one cell per thread instead of two; default 148 = the
 * SM count: 0 forces the two-cell kernel), MMC_COLS_SPLIT=0/1 (one-layer meshes: in-plane pair and z component of the columns
 * kernel in separate CTAs; default: when the grid is below two CTAs per SM). */
int mmc_sweep(mmc_ctx* ctx, int n_sweeps);
/* Same as mmc_sweep, but brackets every phase of every iteration with CUDA events on the ctx stream, synchronises, and
 * returns the summed device time per phase in milliseconds: phase_ms[8] (host) = [0] unused (pack+pad is fused into
 * the rows kernel), [1] rows kernel (S0 + x transform + z-DFT), [2] columns kernel (y transform, tensor multiply S2,
 * inverse y transform), [3] inverse rows kernel (S3, writes B_d), [4] inverse z-DFT pass (several layers only; it runs
 * between [2] and [3]), [5] red pass, [6] black
 * pass, [7] end-of-sweep bookkeeping (on meshes of <= 2^20 cells the last CTA of the black pass
 * does it, so [7] is ~0 there).  Launch-per-kernel with events: the kernels of mmc_sweep, not its graphs. */
int mmc_sweep_timed(mmc_ctx* ctx, int n_sweeps, double* phase_ms);
/* One demag convolution of the current state; bx/by/bz device float[N] (natural order) receive B_d = mu0 H_d
 * in tesla; any of them may be NULL (then the field is only computed).  Works with demag disabled too. */
int mmc_demag_field(mmc_ctx* ctx, float* bx, float* by, float* bz);
/* Synchronises.  E_demag needs the field of the CURRENT state: a convolution is run for it only if the state has changed since
 * the last one (mmc_demag_field, or a previous read-out); the means, counters and running averages never need one. */
int mmc_get_observables(mmc_ctx* ctx, mmc_obs* host_out);
int mmc_reset_counters(mmc_ctx* ctx);                          /* accepted/trials := 0; the cone controller's window is not touched */
int mmc_reset_averages(mmc_ctx* ctx);                          /* run_mean_* := 0 */
/* Histograms of the current state over the non-empty cells, the paper's verification read-outs (PAPER.md:108 length
 * distribution, PAPER.md:114 angular deviation from the mean direction).  kind 0: x = |m|; kind 1: x =
 * polar angle in radians between m and the mean direction (sum of m over the non-empty cells).  nbins (1..4096) equal bins
 * over [lo, hi), bin = floor((x - lo) nbins / (hi - lo)) evaluated in fp64 from the fp32 state; counts: host uint64[nbins];
 * under_over: host uint64[2] (x < lo or NaN, x >= hi), may be NULL.  The paper's solid-angle weighting of the angular
 * histogram is a division by the bin's sin(theta) d(theta) on the caller's side.  Synchronises. */
int mmc_histogram(mmc_ctx* ctx, int kind, int nbins, double lo, double hi, uint64_t* counts, uint64_t* under_over);
/* Chunked convergence of one field step: iterations run in chunks of chunk_sweeps (the paper uses 2000);
 * every chunk's ensemble average of m (mean over the non-empty cells of the state after each iteration, averaged over
 * the chunk) is projected on the unit vector along (ux, uy, uz) -- the applied field direction --; after at least
 * min_chunks (>= 2) chunks the step is accepted when the last two chunk averages differ by at most `threshold` (the
 * paper's "0.01 normalized change": read as an absolute change of <M_par>/Ms0), or given up after max_chunks.
 * The field itself is set with mmc_set_field before the call.  Synchronises once per chunk; uses (and resets) the
 * running averages.  SURVEY 8(f) row 1. */
typedef struct {
    int      chunks_done, converged;
    double   mean_par_last, mean_par_prev;       /* last two chunk averages along the direction */
    double   mean_m[3], mean_len;                /* last chunk's averages */
    uint64_t sweeps;                             /* iterations spent in this call */
} mmc_relax_result;
int mmc_relax(mmc_ctx* ctx, double ux, double uy, double uz, int chunk_sweeps, int min_chunks, int max_chunks,
              double threshold, mmc_relax_result* host_out);
/* One colour pass (colour 0 or 1) at the current sweep counter with a per-cell dump, natural cell order, device
 * pointers, any may be NULL: dm float[3N] (cell-major: dm[3c+a]), dF_terms float[6N] (ex, an, zee, dmi, demag,
 * long in units of kB T), margin float[N] (= ln u - 4 ln f + dF; accept <=> margin < 0), accepted uint8[N].
 * Cells of the other colour and empty cells are left untouched.  The pass updates m like a normal pass, uses the
 * demag field of the last computation, and does not advance the sweep counter. */
int mmc_debug_pass(mmc_ctx* ctx, int colour, float* dm, float* dF_terms, float* margin, uint8_t* accepted);
/* Host-side thermal functions used by the set-up (for tests of the host logic): out[6] = me, chi (1/T), c2, c4,
 * sigma of Eq. (13) with the cap, mu2 = -c2/(2 c4). */
int mmc_thermal(double T, double Tc, double mu_atom, double V, double Ms0, double* out6);
/* Host-side demag tensor used by the set-up: out[6] = N_xx, N_yy, N_zz, N_xy, N_xz, N_yz at integer cell offset. */
int mmc_demag_tensor_at(double dx, double dy, double dz, int ox, int oy, int oz, double* out6);

/* Allocation-free read-out of the magnetisation means, for callers that cannot allocate (stream capture into a CUDA graph,
 * a serving loop, a harness that forbids it): the same sums as the read-out above (<m> and <|m|> over the
 * non-empty cells; |m| rounded to fp32 per cell, fp64 accumulation) by a variant of its kernel whose per-block partial sums
 * sit in a file-scope `static __device__` array of the library instead of a buffer the ctx allocated.  No ctx is needed and
 * the call makes no cudaMalloc / cudaFree / allocating library call, does not synchronise, and only enqueues on cuda_stream
 * (a 256-byte memset node + one kernel), so it may be issued while that stream is being captured.
 *   mx, my, mz : device float[n_cells] on `device`, natural cell order as the state getter returns them (empty cells hold 0:
 *                a cell counts as non-empty when its |m| > 0 -- a non-empty cell never has length 0, see MMC_E_ZERO_LENGTH).
 *   out5       : device double[5] on `device`: <mx>, <my>, <mz>, <|m|> over the non-empty cells, and their number (all 0
 *                when there is none).  Valid once the work enqueued on cuda_stream has run.  Caller-owned, like the inputs.
 *   n_cells    : 0 <= n_cells <= MMC_STATIC_MAX_CELLS; more returns MMC_E_TOO_LARGE and enqueues nothing.  n_cells == 0
 *                only does the set-up below and zeroes out5 (which may then be NULL).
 * Scratch: MMC_STATIC_SCRATCH_BYTES (one 256-byte control line + 5 doubles per block of 4096 cells) of device memory that every
 * GPU which loads the library holds until the process exits.  Its device address is resolved once per device (first call
 * on that device, cudaGetSymbolAddress with the device current; loads the module if CUDA loads lazily): make that first call
 * outside a stream capture.  ALL calls on a device share the array and it keeps the previous call's contents; the call
 * clears what must start at zero (the completion ticket).  Two calls that overlap on the GPU (different streams, or graphs
 * replayed side by side) RACE on it: order them on one stream or with events.  The result does not depend on the
 * schedule of the blocks (fixed summation order).  Errors: MMC_E_INVALID (NULL pointer, n_cells < 0, device < 0 or >= 64),
 * MMC_E_TOO_LARGE, MMC_E_CUDA (the runtime refused the symbol look-up, the memset or the launch). */
#define MMC_STATIC_MAX_CELLS     16777216LL            /* 2^24 cells = 4096 blocks of 4096 cells (config 4 of BASELINE.json: 2^22) */
#define MMC_STATIC_SCRATCH_BYTES (256 + 4096 * 5 * 8)  /* 164 096 bytes */
int mmc_mean_m_static(const float* mx, const float* my, const float* mz, long long n_cells, double* out5,
                      int device, void* cuda_stream);

const char* mmc_strerror(int code);
const char* mmc_last_error(const mmc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MMC_H_ */
