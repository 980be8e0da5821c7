// mmc_internal.h -- declarations shared by the translation units of libmmc_b200 (not part of the ABI).
#ifndef MMC_INTERNAL_H_
#define MMC_INTERNAL_H_

#include <stdint.h>
#include <vector_types.h>
#ifdef __CUDACC__
#include <cuda_runtime.h>
#endif

#include <string>
#include <vector>

#include "../../include/mmc.h"

namespace mmc {

constexpr double kBoltzmann = 1.380649e-23;            // J/K
constexpr double kMu0 = 1.25663706212e-6 * 1.0;        // T m/A  (4 pi 1e-7 to the CODATA-2018 digits)
constexpr int kNearRadius = 40;                        // cells: Newell (binary128) inside, moment expansion beyond

struct ThermalCoef { double me, chi, c2, c4, mu2, sigma13; };
int thermal_coefficients(double T, double Tc, double mu, double V, double Ms0, ThermalCoef* out);
int demag_tensor_at(double dx, double dy, double dz, int ox, int oy, int oz, int r_near, double out[6]);
void demag_tensor_octant(int nx, int ny, int nz, double dx, double dy, double dz, int r_near, std::vector<double> out[6]);

// ---------------------------------------------------------------------------------------------
// Device-side data layout.
// Colour-split storage: cell (i,j,k) of colour col = (i+j+k)&1 lives at
//     col*H + (k*ny + j)*hx + (i>>1),      hx = ceil(nx/2) rounded up to a multiple of 4,  H = hx*ny*nz
// for every per-cell array (m, B_d, mask, per-cell coefficients).  A colour pass then streams its own
// colour densely and reads the other colour as neighbours; no sector carries unused cells.
// ---------------------------------------------------------------------------------------------
struct Geometry {
    int nx, ny, nz;
    int hx;                 // compact row length
    int64_t H;              // cells per colour plane (padded)
    unsigned pbc;
};

// Coefficients of dF/kBT.  Uniform mode: used as they are.  Per-cell mode: kx..gy hold the value at
// T = 1 K and are multiplied by the cell's 1/T; the rest comes from the per-cell arrays.
struct Coef {
    float kx, ky, kz;       // beta * 2 A0 V / h_d^2
    float gx, gy;           // beta * D0 V / dx, beta * D0 V / dy   (DMI, Eq. (15))
    float bKq;              // beta * V * K1 * me
    float bzee;             // beta * V * Ms0
    float c4;               // longitudinal quartic coefficient (units of kB T)
    float sigma;            // length-move half-width
    float ax, ay, az;       // easy axis
    double mu2;             // -c2/(2 c4)  (= me^2 below Tc)
    float Bx, By, Bz;       // applied field, tesla
    float bK1c, bK2c;       // beta V K1c me^10, beta V K2c me^21  (cubic anisotropy, Eq. (12))
    float cub[9];           // the three orthonormal cubic axes
    float bK2u;             // beta V K2 me^6 = beta V K2(T) / me^4  (4th-order uniaxial term of Eq. (11))
};

// Per-cell mode (more than one coefficient class, e.g. cfg 4: one class per distinct (region, T) pair): every cell
// carries one 32-bit word  cw = class << 7 | mask byte  (colour-split, 2*H entries), and the coefficients of a
// class sit in a table of kClassFloats floats per class (48 B = three 16-byte loads); cubic anisotropy adds a second
// table of the same stride, so that meshes without it keep the small footprint in L2.  The table is a few MB for
// the paper's granular film and stays L2-resident; the HBM cost per cell is the 4-byte word.
constexpr int kClassFloats = 12;      // three 16-byte loads per class and table (main table; cubic table only with F_CUBIC)
enum ClassSlot { CS_INVT = 0, CS_C4 = 1, CS_MU2 = 2 /* double in slots 2,3 */, CS_BKQ = 4, CS_BZEE = 5, CS_SIGMA = 6,
                 CS_AX = 7, CS_AY = 8, CS_AZ = 9, CS_K1T = 10 /* beta V K1(T), read-out only */,
                 CS_C0 = 11 /* c0 - c4 mu2^2, read-out only */,
                 /* second table (cubic anisotropy), same stride: */ CS_BK1C = 0, CS_BK2C = 1, CS_CUB = 2 /* 9 floats */, CS_BK2U = 11 };
constexpr unsigned kMaxClasses = 1u << 25;
constexpr float kSumScale = 4194304.f;              // 2^22: fixed-point scale of the running sums (a warp's sum fits int32 for |m| < 8; blocks add in 64 bits)

// Device-resident control block: read by the kernels, advanced by end_sweep_kernel (no host round trip).
struct Control {
    unsigned long long sweep;        // Philox counter word
    unsigned long long accepted, trials;
    unsigned long long win_accepted, win_trials;
    unsigned int win_sweeps;
    int adaptive;
    double cone_deg;
    float one_minus_cos_cone;
    unsigned int pad;                // ticket counter of finish_sweep_ticket (kernels_sweep.cu); 0 between passes
    unsigned long long run_sweeps;   // sweeps accumulated into the running sums
};

enum Feature : unsigned {
    F_MASK = 1u,      // bond/active byte per cell (open boundaries, empty cells, region boundaries)
    F_PERCELL = 2u,   // per-cell coefficient arrays
    F_Z = 4u,         // nz > 1
    F_DMI = 8u,
    F_DEMAG = 16u,
    F_DENSE = 32u,
    F_CUBIC = 64u,    // higher-order anisotropy: cubic, Eq. (12), and the K2 term of Eq. (11) (second class table)    // no empty cell: every in-mesh cell is active, so no load has to wait for the mask / class word
};

struct SweepArgs {
    Geometry g;
    float* m[3];                 // colour-split
    const float* bd[3];          // colour-split B_d (tesla) or NULL
    const uint8_t* mask;         // colour-split; bits 0..5 bonded +x,-x,+y,-y,+z,-z; bit 6 active
    const uint32_t* cw;          // per-cell mode: class << 7 | mask (colour-split), else NULL
    const float4* table;         // per-cell mode: kClassFloats floats per class, else NULL
    const float4* table_cubic;   // per-cell mode with cubic anisotropy: kClassFloats floats per class (CS_BK1C ...), else NULL
    Coef coef;
    Control* ctl;
    unsigned seed_lo, seed_hi;
    int colour;
    int finish;                  // != 0: the last CTA of this pass runs the end-of-sweep bookkeeping (S11) itself
    int pass1_below;              // host side only: grids of fewer CTAs take the one-cell-per-thread pass kernel (launch_colour_pass)
    unsigned long long* run_sums; // [4] running sums of the sweeps' final mx,my,mz,|m| in fixed point (two's complement, kSumScale), or NULL
    // debug dump (natural order), any NULL
    float* dbg_dm; float* dbg_terms; float* dbg_margin; uint8_t* dbg_acc;
};

struct Observables { double sum[4]; double E[6]; unsigned long long n_active; };
// What one read-out brings to the host, gathered by the read-out kernel so that it is ONE device-to-host copy (into pinned memory)
struct ReadOut { Observables obs; Control ctl; unsigned long long run_sums[4]; };

// TMA-staged colour pass (kernels_sweep.cu): tensor maps (CUtensorMap is 128 bytes, 64-byte aligned) over the colour-split
// arrays as rank-4 tensors (x = compact index, y, z, colour) and the tile shape they were encoded for.
struct alignas(64) PassTmaMaps { unsigned char own_m[3][128], oth_m[3][128], bd[3][128], cw[128]; };
struct PassTmaShape { int BY, BZ, zh, tiles_x, tiles_y, tiles_z, oth_arr, oth_box_bytes; };
struct PassTma {
    bool ok = false;
    PassTmaShape sh{};
    PassTmaMaps maps{};
    const void* key[3] = { nullptr, nullptr, nullptr };   // m[0], bd[0], cw the maps were built for
};
// builds the maps when the mesh qualifies (no periodic direction, driver entry point available); ok = false otherwise
void pass_tma_build(const Geometry& g, float* const m[3], float* const bd[3], const uint32_t* cw, PassTma* out);

// kernels_sweep.cu
int launch_colour_pass(const SweepArgs& a, unsigned features, bool debug, void* stream, const PassTma* tma = nullptr);
int launch_end_sweep(Control* ctl, void* stream);
int launch_small_mesh_sweeps(const SweepArgs& a, unsigned features, int n_sweeps, void* stream);
// kernels_layout.cu
int launch_to_split(const Geometry& g, const float* nat, float* split, void* stream);
int launch_from_split(const Geometry& g, const float* split, float* nat, void* stream);
int launch_check_state(const Geometry& g, float* const m[3], const uint8_t* mask, int* flag, void* stream);
struct ObsParams {
    float K1T_u;                           // beta V K1(T), uniform mode (units of kB T); per-cell mode: class table
    float c0_u;                            // c0 - c4 mu2^2, uniform mode (units of kB T)
    double aex[3];                         // A0 V / h_d^2 (joule)
    double D0V;                            // D0 V (J m)
    double inv_d[2];                       // 1/dx, 1/dy
    double kB;
    float T_u;                             // uniform temperature (per-cell mode reads 1/T per cell)
};
int launch_observables(const SweepArgs& a, bool percell, const ObsParams& op, ReadOut* dev_out, double* scratch,
                       int scratch_blocks, void* stream);

int launch_histogram(const Geometry& g, const float* const m[3], const uint8_t* mask, int kind, const double dir[3], int nbins,
                     double lo, double hi, unsigned long long* dev_counts, void* stream);

// Optional per-phase device timing (mmc_sweep_timed): mark(p) records an event that ends phase p.
enum Phase { PH_PACK = 0, PH_FFT_FWD, PH_MULTIPLY, PH_FFT_INV, PH_CROP, PH_RED, PH_BLACK, PH_END, PH_COUNT };
struct PhaseTimer {
    std::vector<void*> events;     // cudaEvent_t
    std::vector<int> phase;        // phase ended by events[i]; -1 = start marker
    bool failed = false;           // an event could not be created / recorded: the phase times would be wrong
    void mark(int ph, void* stream);
};

// demag.cu
struct DemagPlan;
int demag_create(DemagPlan** out, const Geometry& g, double dx, double dy, double dz, void* stream, std::string* err);
void demag_destroy(DemagPlan* p);
// Ms0 (colour-split, A/m per cell, 0 in empty cells) times m -> B_d colour-split (tesla)
int demag_compute(DemagPlan* p, const float* const m[3], const float* Ms0_split, float Ms0_uniform,
                  float* const bd[3], void* stream, std::string* err, PhaseTimer* timer = nullptr);

#ifdef __CUDACC__
// Programmatic dependent launch (PDL), an option (MMC_PDL=1).  Every kernel of the iteration path starts with pdl_enter():
// it lets the NEXT kernel of the stream be launched right away (its CTAs become resident as slots free up and park in
// griddepcontrol.wait) and then waits until the PREVIOUS kernel has completed and flushed its memory, before it reads or writes
// anything; the kernels are launched with launch_pdl (programmatic stream serialisation allowed when g_pdl is set), in streams
// and in captured graphs alike.  Measured (round 2): bit-identical results, but SLOWER on every config (the parked CTAs take
// slots from the running kernel), so g_pdl is off by default and pdl_enter() is then a pair of no-ops.
extern bool g_pdl;
__device__ __forceinline__ void pdl_enter()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
template <class... P, class... A>
inline cudaError_t launch_pdl(void (*kern)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A&&... args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = g_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<P>(args)...);
}
#endif

}  // namespace mmc

#endif
