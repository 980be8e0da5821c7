// api.cu -- the extern "C" boundary of include/mmc.h: context, host-side set-up (thermal classes, bond/active
// mask, coefficient upload), the iteration loop (demag -> red -> black -> end_sweep) and the read-outs.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <unordered_map>

#include "mmc_internal.h"

using namespace mmc;

namespace mmc { bool g_pdl = false; }     // see mmc_internal.h, launch_pdl

struct mmc_ctx {
    Geometry g{};
    double dx = 0, dy = 0, dz = 0, V = 0;
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    // problem description (host)
    std::vector<mmc_material> regions;
    std::vector<int32_t> region_of_cell;          // empty => all 0
    int inter_region = 1;
    double T_uniform = 0.0; std::vector<float> T_cell;   // T_cell empty => uniform
    bool T_set = false, material_set = false, m_set = false;
    double B[3] = { 0, 0, 0 };
    double cone_deg = 30.0, sigma_user = -1.0; int adaptive = 0;
    int demag_enabled = 0, demag_updates = 1;
    uint64_t seed = 0;
    // derived (host)
    bool dirty = true, m_needs_check = false;
    // B_d bookkeeping: state_version counts every change of m (or of Ms0), bd_version is the state_version whose field sits in
    // bd[] (0 = none): a read-out or the first iteration of a sweep does not repeat a convolution of an unchanged state
    uint64_t state_version = 1, bd_version = 0;
    // CUDA graphs of whole iterations (launch-per-kernel path): kernel arguments are captured by value, so the graphs are
    // rebuilt whenever a setter changes anything a launch depends on (args_version); device-side state (m, control block,
    // sweep counter) is read through pointers and needs no rebuild.  Captured on a private stream (the caller's stream may
    // be the legacy default stream, which cannot be captured) and launched into the caller's stream.
    uint64_t args_version = 1;
    struct IterGraph { cudaGraphExec_t exec = nullptr; uint64_t version = 0; };
    IterGraph graph1, graphN;
    cudaStream_t cap_stream = nullptr;
    bool graphs_off = false;
    PassTma tma;                                  // TMA-staged pass: tensor maps over m, bd, cw (rebuilt when a pointer changes)
    bool tma_off = false;
    int pass1_below = 148;                        // MMC_PASS1_BELOW: see launch_colour_pass
    bool percell = false;
    unsigned features = 0;
    double A0 = 0, D0 = 0, sigma_first = 0;
    Coef coef{};
    float K1T_u = 0.f, c0_u = 0.f, Ms0_u = 0.f;
    bool Ms0_uniform = true;
    unsigned long long n_active = 0;
    // device
    float* m[3] = { nullptr, nullptr, nullptr };
    float* bd[3] = { nullptr, nullptr, nullptr };
    // every uploaded buffer carries its own capacity (elements); upload() grows it when needed
    uint8_t* mask = nullptr; size_t mask_cap = 0;
    float* Ms0_split = nullptr; size_t ms0_cap = 0;
    uint32_t* cw = nullptr; size_t cw_cap = 0;    // per-cell mode: class << 7 | mask (colour-split)
    float* table = nullptr; size_t table_cap = 0; // per-cell mode: kClassFloats floats per class
    float* table_cubic = nullptr; size_t table_cubic_cap = 0;   // ... and the cubic-anisotropy table of the same stride
    size_t n_classes = 0;
    Control* ctl = nullptr;
    unsigned long long* run_sums = nullptr;       // [4] fixed-point running sums (kSumScale)
    double* obs_scratch = nullptr; int obs_blocks = 0;
    ReadOut* d_obs = nullptr;                     // device: filled by the read-out kernel
    ReadOut* h_obs = nullptr;                     // pinned host: target of the one copy of a read-out
    int* d_flag = nullptr;
    float* stage = nullptr;                       // N floats, for natural-order outputs
    DemagPlan* demag = nullptr;
};

namespace {

int fail(mmc_ctx* c, int code, const std::string& msg) { if (c) c->err = msg; return code; }

#define CU(c, x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return fail((c), MMC_E_CUDA, std::string(#x) + ": " + cudaGetErrorString(e_)); } while (0)

struct DeviceGuard {
    int prev = -1; bool ok;
    explicit DeviceGuard(int dev) { ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline long long split_index_h(const Geometry& g, int i, int j, int k)
{
    const int col = (i + j + k) & 1;
    return (long long)col * g.H + ((long long)k * g.ny + j) * g.hx + (i >> 1);
}

// Host vector -> device buffer that grows to fit: *cap is the allocation of *dptr in elements (0 = none).  A buffer is
// never written beyond its own allocation, whatever the order of set_material / set_temperature calls on a long-lived ctx.
template <class T>
int upload(mmc_ctx* c, T** dptr, size_t* cap, const std::vector<T>& h)
{
    if (h.empty()) return MMC_OK;
    if (h.size() > *cap) {
        CU(c, cudaStreamSynchronize(c->stream));     // kernels in flight may still read the old buffer
        cudaFree(*dptr); *dptr = nullptr; *cap = 0;
        if (cudaMalloc(dptr, h.size() * sizeof(T)) != cudaSuccess) { *dptr = nullptr; return fail(c, MMC_E_NOMEM, "device allocation failed"); }
        *cap = h.size();
    }
    CU(c, cudaMemcpyAsync(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return MMC_OK;
}

// O1 + mask: everything the kernels need that depends on material, temperature, move and coupling settings.
int ensure_setup(mmc_ctx* c)
{
    if (!c->dirty) return MMC_OK;
    const Geometry& g = c->g;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const size_t S = (size_t)(2 * g.H);
    const bool have_reg = !c->region_of_cell.empty();
    const int nreg = (int)c->regions.size();
    // uniform exchange / DMI constants over non-empty regions
    bool any = false; double A0 = 0, D0 = 0;
    for (const auto& r : c->regions) {
        if (!(r.Ms0 > 0)) continue;
        if (!any) { A0 = r.A0; D0 = r.D0; any = true; }
        else if (r.A0 != A0 || r.D0 != D0) return fail(c, MMC_E_UNSUPPORTED, "A0 and D0 must be equal in all non-empty regions");
    }
    c->A0 = A0; c->D0 = D0;
    auto reg_of = [&](long long cell) -> int { return have_reg ? c->region_of_cell[cell] : 0; };
    auto T_of = [&](long long cell) -> float { return c->T_cell.empty() ? (float)c->T_uniform : c->T_cell[cell]; };
    // classes = distinct (region, T) pairs among active cells
    struct Cls { int region; float T; ThermalCoef th; };
    std::vector<Cls> classes;
    std::unordered_map<uint64_t, int> cls_of_key;
    std::vector<int> cls_of_cell((size_t)N, -1);
    unsigned long long n_active = 0;
    for (long long cell = 0; cell < N; ++cell) {
        const int r = reg_of(cell);
        if (!(c->regions[r].Ms0 > 0)) continue;
        n_active++;
        const float T = T_of(cell);
        uint32_t tb; std::memcpy(&tb, &T, 4);
        const uint64_t key = ((uint64_t)(uint32_t)r << 32) | tb;
        auto it = cls_of_key.find(key);
        int id;
        if (it == cls_of_key.end()) {
            if (!(T > 0.f) || !std::isfinite(T)) return fail(c, MMC_E_INVALID, "temperature must be > 0 in every non-empty cell");
            Cls k; k.region = r; k.T = T;
            const mmc_material& mt = c->regions[r];
            if (!(mt.Tc > 0) || !(mt.mu_atom > 0)) return fail(c, MMC_E_INVALID, "Tc and mu_atom must be > 0 in non-empty regions");
            int rc = thermal_coefficients((double)T, mt.Tc, mt.mu_atom, c->V, mt.Ms0, &k.th);
            if (rc != MMC_OK) return fail(c, rc, "thermal_coefficients failed");
            id = (int)classes.size(); classes.push_back(k); cls_of_key.emplace(key, id);
        } else id = it->second;
        cls_of_cell[(size_t)cell] = id;
    }
    c->n_active = n_active;
    // per-cell mode iff more than one class differs in anything the kernel reads
    c->percell = classes.size() > 1;
    // mask (bit d: bonded neighbour in direction d; bit 6: active), Ms0
    std::vector<uint8_t> mask(S, 0);
    std::vector<float> ms0(S, 0.f);
    bool need_mask = false;
    bool ms0_uniform = true; double ms0_first = -1;
    const int nn[3] = { g.nx, g.ny, g.nz };
    for (int k = 0; k < g.nz; ++k) for (int j = 0; j < g.ny; ++j) for (int i = 0; i < g.nx; ++i) {
        const long long cell = (long long)i + (long long)g.nx * (j + (long long)g.ny * k);
        const long long s = split_index_h(g, i, j, k);
        if (cls_of_cell[(size_t)cell] < 0) { need_mask = true; continue; }
        const int r = reg_of(cell);
        const double Ms = c->regions[r].Ms0;
        ms0[(size_t)s] = (float)Ms;
        if (ms0_first < 0) ms0_first = Ms; else if (Ms != ms0_first) ms0_uniform = false;
        unsigned mb = 0x40u;
        const int q[3] = { i, j, k };
        for (int d = 0; d < 6; ++d) {
            const int a = d >> 1, step = (d & 1) ? -1 : 1;
            if (nn[a] < 2) continue;
            int v = q[a] + step;
            if (v < 0 || v >= nn[a]) { if (!((g.pbc >> a) & 1u)) { need_mask = true; continue; } v = (v + nn[a]) % nn[a]; }
            int p[3] = { i, j, k }; p[a] = v;
            const long long nb = (long long)p[0] + (long long)g.nx * (p[1] + (long long)g.ny * p[2]);
            if (cls_of_cell[(size_t)nb] < 0) { need_mask = true; continue; }
            if (!c->inter_region && reg_of(nb) != r) { need_mask = true; continue; }
            mb |= 1u << d;
        }
        mask[(size_t)s] = (uint8_t)mb;
    }
    c->Ms0_uniform = ms0_uniform && n_active == (unsigned long long)N;   // empty cells need per-cell weights to zero their M
    c->Ms0_u = ms0_first > 0 ? (float)ms0_first : 0.f;
    int rc = upload(c, &c->mask, &c->mask_cap, mask); if (rc) return rc;
    if (!c->Ms0_uniform) { rc = upload(c, &c->Ms0_split, &c->ms0_cap, ms0); if (rc) return rc; }
    // coefficients
    const double V = c->V, kB = kBoltzmann;
    const double Jd[3] = { 2.0 * A0 * V / (c->dx * c->dx), 2.0 * A0 * V / (c->dy * c->dy), 2.0 * A0 * V / (c->dz * c->dz) };
    Coef cf{};
    cf.Bx = (float)c->B[0]; cf.By = (float)c->B[1]; cf.Bz = (float)c->B[2];
    // one table entry (kClassFloats floats, ClassSlot order) per class
    auto class_values = [&](const Cls& k, double beta, float* out, float* outc) {
        const mmc_material& mt = c->regions[k.region];
        double al = std::sqrt(mt.ax * mt.ax + mt.ay * mt.ay + mt.az * mt.az);
        double ex = 0, ey = 0, ez = 1;
        if (al > 0) { ex = mt.ax / al; ey = mt.ay / al; ez = mt.az / al; }
        const double sig = c->sigma_user >= 0 ? c->sigma_user : k.th.sigma13;
        out[CS_INVT] = (float)(1.0 / (double)k.T); out[CS_C4] = (float)k.th.c4;
        std::memcpy(&out[CS_MU2], &k.th.mu2, sizeof(double));
        out[CS_BKQ] = (float)(beta * V * mt.K1 * k.th.me); out[CS_BZEE] = (float)(beta * V * mt.Ms0); out[CS_SIGMA] = (float)sig;
        out[CS_AX] = (float)ex; out[CS_AY] = (float)ey; out[CS_AZ] = (float)ez;
        out[CS_K1T] = (float)(beta * V * mt.K1 * k.th.me * k.th.me * k.th.me);
        out[CS_C0] = (float)((k.th.me > 0 || k.th.mu2 == 0) ? 0.0 : -k.th.c4 * k.th.mu2 * k.th.mu2);
        // cubic anisotropy: K(T) = K me^(l(l+1)/2), l = 4, 6; axes by Gram-Schmidt, e3 = e1 x e2
        outc[CS_BK1C] = (float)(beta * V * mt.K1c * std::pow(k.th.me, 10.0));
        outc[CS_BK2C] = (float)(beta * V * mt.K2c * std::pow(k.th.me, 21.0));
        outc[CS_BK2U] = (float)(k.th.me > 0 ? beta * V * mt.K2 * std::pow(k.th.me, 6.0) : 0.0);
        double e1[3] = { mt.c1x, mt.c1y, mt.c1z }, e2[3] = { mt.c2x, mt.c2y, mt.c2z };
        double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
        if (!(n1 > 0)) { e1[0] = 1; e1[1] = e1[2] = 0; n1 = 1; }
        for (int q = 0; q < 3; ++q) e1[q] /= n1;
        const double pr = e2[0] * e1[0] + e2[1] * e1[1] + e2[2] * e1[2];
        for (int q = 0; q < 3; ++q) e2[q] -= pr * e1[q];
        double n2 = std::sqrt(e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2]);
        if (!(n2 > 1e-12)) { const int a = std::fabs(e1[0]) < 0.9 ? 0 : 1; e2[0] = e2[1] = e2[2] = 0; e2[a] = 1;   // unused axes: any frame
            const double p2 = e1[a]; for (int q = 0; q < 3; ++q) e2[q] -= p2 * e1[q]; n2 = std::sqrt(e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2]); }
        for (int q = 0; q < 3; ++q) e2[q] /= n2;
        const double e3[3] = { e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0] };
        for (int q = 0; q < 3; ++q) { outc[CS_CUB + q] = (float)e1[q]; outc[CS_CUB + 3 + q] = (float)e2[q]; outc[CS_CUB + 6 + q] = (float)e3[q]; }
    };
    c->n_classes = classes.size();
    if (!c->percell) {
        if (!classes.empty()) {
            const Cls& k = classes[0];
            const double beta = 1.0 / (kB * (double)k.T);
            float v[kClassFloats], vc[kClassFloats];
            class_values(k, beta, v, vc);
            cf.kx = (float)(beta * Jd[0]); cf.ky = (float)(beta * Jd[1]); cf.kz = (float)(beta * Jd[2]);
            cf.gx = (float)(beta * D0 * V / c->dx); cf.gy = (float)(beta * D0 * V / c->dy);
            cf.c4 = v[CS_C4]; cf.mu2 = k.th.mu2; cf.bKq = v[CS_BKQ]; cf.bzee = v[CS_BZEE]; cf.sigma = v[CS_SIGMA];
            cf.ax = v[CS_AX]; cf.ay = v[CS_AY]; cf.az = v[CS_AZ];
            cf.bK1c = vc[CS_BK1C]; cf.bK2c = vc[CS_BK2C];
            for (int q = 0; q < 9; ++q) cf.cub[q] = vc[CS_CUB + q];
            cf.bK2u = vc[CS_BK2U];
            c->K1T_u = v[CS_K1T]; c->c0_u = v[CS_C0];
            c->sigma_first = v[CS_SIGMA];
        }
    } else {
        if (classes.size() > (size_t)kMaxClasses) return fail(c, MMC_E_UNSUPPORTED, "more than 2^25 distinct (region, T) classes");
        const double b1 = 1.0 / kB;                   // beta at T = 1 K; the kernel multiplies by the class's 1/T
        cf.kx = (float)(b1 * Jd[0]); cf.ky = (float)(b1 * Jd[1]); cf.kz = (float)(b1 * Jd[2]);
        cf.gx = (float)(b1 * D0 * V / c->dx); cf.gy = (float)(b1 * D0 * V / c->dy);
        std::vector<float> tab(classes.size() * kClassFloats), tabc(classes.size() * kClassFloats);
        for (size_t q = 0; q < classes.size(); ++q)
            class_values(classes[q], 1.0 / (kB * (double)classes[q].T), &tab[kClassFloats * q], &tabc[kClassFloats * q]);
        c->sigma_first = tab[CS_SIGMA];
        rc = upload(c, &c->table, &c->table_cap, tab); if (rc) return rc;
        bool cubic = false;
        for (const auto& r : c->regions) if (r.Ms0 > 0 && (r.K1c != 0.0 || r.K2c != 0.0 || r.K2 != 0.0)) cubic = true;
        if (cubic) { rc = upload(c, &c->table_cubic, &c->table_cubic_cap, tabc); if (rc) return rc; }
        std::vector<uint32_t> cw(S, 0u);
        for (int k = 0; k < g.nz; ++k) for (int j = 0; j < g.ny; ++j) for (int i = 0; i < g.nx; ++i) {
            const long long cell = (long long)i + (long long)g.nx * (j + (long long)g.ny * k);
            const int id = cls_of_cell[(size_t)cell];
            const size_t sidx = (size_t)split_index_h(g, i, j, k);
            if (id >= 0) cw[sidx] = ((uint32_t)id << 7) | mask[sidx];
        }
        rc = upload(c, &c->cw, &c->cw_cap, cw); if (rc) return rc;
    }
    c->coef = cf;
    unsigned f = 0;
    if (need_mask) f |= F_MASK;
    if (c->percell) f |= F_PERCELL;
    if (g.nz > 1) f |= F_Z;
    if (D0 != 0.0) f |= F_DMI;
    if (c->demag_enabled) f |= F_DEMAG;
    if (n_active == (unsigned long long)N) f |= F_DENSE;
    for (const auto& r : c->regions)
        if (r.Ms0 > 0 && (r.K1c != 0.0 || r.K2c != 0.0 || r.K2 != 0.0)) f |= F_CUBIC;
    c->features = f;
    c->tma.ok = false;
    // TMA boxes bring in whole tiles, empty cells included, while the brick kernel skips the loads of empty cells: staged only
    // for meshes that are mostly magnetic (BASELINE config 5 is 30 % magnetic and loses 5 % with staging, measured)
    if (!c->tma_off && n_active * 10ull >= (unsigned long long)N * 6ull) pass_tma_build(c->g, c->m, c->bd, c->percell ? c->cw : nullptr, &c->tma);
    c->dirty = false;
    c->bd_version = 0;                                   // Ms0 or the set of non-empty cells may have changed
    return MMC_OK;
}

int push_control(mmc_ctx* c, bool reset_window)
{
    Control h;
    CU(c, cudaMemcpyAsync(&h, c->ctl, sizeof(Control), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    h.adaptive = c->adaptive; h.cone_deg = c->cone_deg;
    const double s = std::sin(0.5 * c->cone_deg * 0.017453292519943295);
    h.one_minus_cos_cone = (float)(2.0 * s * s);
    if (reset_window) { h.accepted += h.win_accepted; h.trials += h.win_trials; h.win_accepted = h.win_trials = 0; h.win_sweeps = 0; }
    CU(c, cudaMemcpyAsync(c->ctl, &h, sizeof(Control), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return MMC_OK;
}

SweepArgs make_args(mmc_ctx* c, int colour)
{
    SweepArgs a{};
    a.g = c->g;
    for (int q = 0; q < 3; ++q) { a.m[q] = c->m[q]; a.bd[q] = c->bd[q]; }
    a.mask = c->mask; a.coef = c->coef;
    a.coef.Bx = (float)c->B[0]; a.coef.By = (float)c->B[1]; a.coef.Bz = (float)c->B[2];
    a.cw = c->percell ? c->cw : nullptr; a.table = c->percell ? reinterpret_cast<const float4*>(c->table) : nullptr;
    a.table_cubic = (c->percell && (c->features & F_CUBIC)) ? reinterpret_cast<const float4*>(c->table_cubic) : nullptr;
    a.ctl = c->ctl; a.seed_lo = (unsigned)c->seed; a.seed_hi = (unsigned)(c->seed >> 32);
    a.colour = colour; a.run_sums = c->run_sums; a.pass1_below = c->pass1_below;
    return a;
}

int ensure_demag(mmc_ctx* c)
{
    if (c->demag) return MMC_OK;
    std::string e;
    int rc = demag_create(&c->demag, c->g, c->dx, c->dy, c->dz, c->stream, &e);
    if (rc != MMC_OK) { demag_destroy(c->demag); c->demag = nullptr; return fail(c, rc, "demag set-up: " + e); }
    return MMC_OK;
}

int compute_demag(mmc_ctx* c, PhaseTimer* timer = nullptr, cudaStream_t stream_override = nullptr, bool use_override = false)
{
    int rc = ensure_demag(c); if (rc) return rc;
    std::string e;
    rc = demag_compute(c->demag, c->m, c->Ms0_uniform ? nullptr : c->Ms0_split, c->Ms0_u, c->bd, use_override ? stream_override : c->stream, &e, timer);
    if (rc != MMC_OK) { c->bd_version = 0; return fail(c, rc, "demag: " + e); }
    c->bd_version = c->state_version;
    return MMC_OK;
}

int check_m(mmc_ctx* c)
{
    CU(c, cudaMemsetAsync(c->d_flag, 0, sizeof(int), c->stream));
    int rc = launch_check_state(c->g, c->m, c->mask, c->d_flag, c->stream);
    if (rc) return fail(c, rc, "check_state launch failed");
    int flag = 0;
    CU(c, cudaMemcpyAsync(&flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    c->m_needs_check = false;
    c->state_version++;
    if (flag & 1) return fail(c, MMC_E_ZERO_LENGTH, "a non-empty cell has zero (or non-finite) magnetisation");
    if (flag & 2) return fail(c, MMC_E_INVALID, "a non-empty cell has |m| >= 2: m is M/Ms0 (PAPER.md:32), not M in A/m");
    return MMC_OK;
}

int ready(mmc_ctx* c)
{
    if (!c) return MMC_E_INVALID;
    if (!c->material_set || !c->T_set || !c->m_set) return fail(c, MMC_E_STATE, "set material, temperature and m before this call");
    int rc = ensure_setup(c); if (rc) return rc;
    if (c->m_needs_check) { rc = check_m(c); if (rc) return rc; }
    return MMC_OK;
}

}  // namespace

extern "C" {

int mmc_create(mmc_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz, unsigned pbc_mask, int device, void* cuda_stream)
{
    if (!out) return MMC_E_INVALID;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || pbc_mask > 7u) return MMC_E_INVALID;
    if (2ll * ((((nx + 1) / 2) + 3) / 4 * 4) * ny * nz >= (1ll << 31)) return MMC_E_INVALID;   // kernels use 32-bit element offsets
    const int nn[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a)
        if (((pbc_mask >> a) & 1u) && (nn[a] < 2 || (nn[a] & 1))) return MMC_E_INVALID;   // checkerboard needs even periodic lengths
    mmc_ctx* c = new (std::nothrow) mmc_ctx();
    if (!c) return MMC_E_NOMEM;
    c->g.nx = nx; c->g.ny = ny; c->g.nz = nz; c->g.pbc = pbc_mask;
    c->g.hx = (((nx + 1) / 2) + 3) / 4 * 4;
    c->g.H = (int64_t)c->g.hx * ny * nz;
    c->dx = dx; c->dy = dy; c->dz = dz; c->V = dx * dy * dz;
    c->device = device; c->stream = (cudaStream_t)cuda_stream;
    c->graphs_off = std::getenv("MMC_NO_GRAPH") != nullptr;      // A/B knob: plain launches only
    // programmatic dependent launch between the kernels of an iteration: measured slower on every config (early-resident CTAs of
    // the next kernel take slots from the running one: cfg 2 26.5 against 23.2 us, cfg 4 0.584 against 0.497 ms), so it is off
    // unless MMC_PDL=1 (process-wide knob, read at every create)
    { const char* e = std::getenv("MMC_PDL"); mmc::g_pdl = e && e[0] == '1'; }
    { const char* e = std::getenv("MMC_PASS1_BELOW"); if (e) c->pass1_below = std::atoi(e); }
    // the TMA-staged pass runs at the speed of the L1-served brick kernel on the meshes it serves (both
    // ncu tables in profiles/): the brick kernel, which serves every mesh, is the default; MMC_TMA=1 selects the staged variant
    { const char* e = std::getenv("MMC_TMA"); c->tma_off = !(e && e[0] == '1'); }
    c->regions.push_back(mmc_material{ 0, 0, 0, 0, 0, 1, 0, 1, 9.2740100783e-24, 0, 0, 1, 0, 0, 0, 1, 0, 0 });
    DeviceGuard dg(device);
    auto bail = [&](int code) { mmc_destroy(c); return code; };
    if (!dg.ok) return bail(MMC_E_CUDA);
    const size_t S = (size_t)(2 * c->g.H);
    for (int q = 0; q < 3; ++q) {
        if (cudaMalloc(&c->m[q], S * sizeof(float)) != cudaSuccess) return bail(MMC_E_NOMEM);
        if (cudaMalloc(&c->bd[q], S * sizeof(float)) != cudaSuccess) return bail(MMC_E_NOMEM);
        cudaMemsetAsync(c->m[q], 0, S * sizeof(float), c->stream);
        cudaMemsetAsync(c->bd[q], 0, S * sizeof(float), c->stream);
    }
    c->obs_blocks = 148 * 20;                     // 128-thread CTAs (kernels_layout.cu), five per SM: four whole waves; ~11 slots per thread on the 4 M-cell meshes
    if (cudaMalloc(&c->ctl, sizeof(Control)) != cudaSuccess) return bail(MMC_E_NOMEM);
    if (cudaMalloc(&c->run_sums, 4 * sizeof(unsigned long long)) != cudaSuccess) return bail(MMC_E_NOMEM);
    if (cudaMalloc(&c->obs_scratch, ((size_t)c->obs_blocks * 11 + 1) * sizeof(double)) != cudaSuccess) return bail(MMC_E_NOMEM);   // ticket + partials
    if (cudaMalloc(&c->d_obs, sizeof(ReadOut)) != cudaSuccess) return bail(MMC_E_NOMEM);
    if (cudaHostAlloc(&c->h_obs, sizeof(ReadOut), cudaHostAllocDefault) != cudaSuccess) return bail(MMC_E_NOMEM);
    cudaMemsetAsync(c->obs_scratch, 0, sizeof(double), c->stream);      // the read-out kernel's ticket
    if (cudaMalloc(&c->d_flag, sizeof(int)) != cudaSuccess) return bail(MMC_E_NOMEM);
    if (cudaMalloc(&c->stage, (size_t)nx * ny * nz * sizeof(float)) != cudaSuccess) return bail(MMC_E_NOMEM);
    cudaMemsetAsync(c->ctl, 0, sizeof(Control), c->stream);
    cudaMemsetAsync(c->run_sums, 0, 4 * sizeof(unsigned long long), c->stream);
    if (push_control(c, false) != MMC_OK) return bail(MMC_E_CUDA);
    *out = c;
    return MMC_OK;
}

int mmc_destroy(mmc_ctx* c)
{
    if (!c) return MMC_E_INVALID;
    DeviceGuard dg(c->device);
    cudaStreamSynchronize(c->stream);
    for (int q = 0; q < 3; ++q) { cudaFree(c->m[q]); cudaFree(c->bd[q]); }
    cudaFree(c->cw); cudaFree(c->table); cudaFree(c->table_cubic);
    cudaFree(c->mask); cudaFree(c->Ms0_split); cudaFree(c->ctl); cudaFree(c->run_sums); cudaFree(c->obs_scratch);
    cudaFree(c->d_obs); cudaFreeHost(c->h_obs); cudaFree(c->d_flag); cudaFree(c->stage);
    demag_destroy(c->demag);
    if (c->graph1.exec) cudaGraphExecDestroy(c->graph1.exec);
    if (c->graphN.exec) cudaGraphExecDestroy(c->graphN.exec);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    delete c;
    return MMC_OK;
}

int mmc_set_material(mmc_ctx* c, int n_regions, const mmc_material* regions, const int32_t* region_of_cell)
{
    if (!c) return MMC_E_INVALID;
    if (n_regions < 1 || !regions) return fail(c, MMC_E_INVALID, "n_regions >= 1 and regions != NULL required");
    for (int r = 0; r < n_regions; ++r)
        if (!(regions[r].Ms0 >= 0) || !std::isfinite(regions[r].Ms0) || regions[r].A0 < 0) return fail(c, MMC_E_INVALID, "Ms0 and A0 must be >= 0");
    for (int r = 0; r < n_regions; ++r) {
        const mmc_material& mt = regions[r];
        if (mt.K1c == 0.0 && mt.K2c == 0.0) continue;
        const double cx = mt.c1y * mt.c2z - mt.c1z * mt.c2y, cy = mt.c1z * mt.c2x - mt.c1x * mt.c2z, cz = mt.c1x * mt.c2y - mt.c1y * mt.c2x;
        const double n1 = mt.c1x * mt.c1x + mt.c1y * mt.c1y + mt.c1z * mt.c1z, n2 = mt.c2x * mt.c2x + mt.c2y * mt.c2y + mt.c2z * mt.c2z;
        if (!(cx * cx + cy * cy + cz * cz > 1e-12 * n1 * n2)) return fail(c, MMC_E_INVALID, "cubic axes c1, c2 must not be parallel or zero");
    }
    const long long N = (long long)c->g.nx * c->g.ny * c->g.nz;
    if (region_of_cell)
        for (long long i = 0; i < N; ++i)
            if (region_of_cell[i] < 0 || region_of_cell[i] >= n_regions) return fail(c, MMC_E_INVALID, "region_of_cell out of range");
    c->regions.assign(regions, regions + n_regions);
    if (region_of_cell) c->region_of_cell.assign(region_of_cell, region_of_cell + N); else c->region_of_cell.clear();
    c->material_set = true; c->dirty = true; c->m_needs_check = c->m_set; c->args_version++;
    return MMC_OK;
}

int mmc_set_exchange_coupling(mmc_ctx* c, int inter_region_exchange)
{
    if (!c) return MMC_E_INVALID;
    c->inter_region = inter_region_exchange ? 1 : 0; c->dirty = true; c->args_version++;
    return MMC_OK;
}

int mmc_set_temperature(mmc_ctx* c, double T_uniform, const float* T_per_cell)
{
    if (!c) return MMC_E_INVALID;
    const long long N = (long long)c->g.nx * c->g.ny * c->g.nz;
    if (T_per_cell) {
        c->T_cell.assign(T_per_cell, T_per_cell + N);
    } else {
        if (!(T_uniform > 0) || !std::isfinite(T_uniform)) return fail(c, MMC_E_INVALID, "T must be > 0");
        c->T_cell.clear();
    }
    c->T_uniform = T_uniform; c->T_set = true; c->dirty = true; c->args_version++;
    return MMC_OK;
}

int mmc_set_field(mmc_ctx* c, double Bx, double By, double Bz)
{
    if (!c) return MMC_E_INVALID;
    if (!std::isfinite(Bx) || !std::isfinite(By) || !std::isfinite(Bz)) return fail(c, MMC_E_INVALID, "field must be finite");
    c->B[0] = Bx; c->B[1] = By; c->B[2] = Bz; c->args_version++;          // read into the kernel arguments at every launch
    return MMC_OK;
}

int mmc_set_move(mmc_ctx* c, double cone_deg, double sigma, int adaptive_cone)
{
    if (!c) return MMC_E_INVALID;
    if (!(cone_deg > 0) || cone_deg > 180.0 || !(sigma < 1.0)) return fail(c, MMC_E_INVALID, "0 < cone <= 180 and sigma < 1 required");
    c->cone_deg = cone_deg; c->sigma_user = sigma; c->adaptive = adaptive_cone ? 1 : 0; c->dirty = true; c->args_version++;
    DeviceGuard dg(c->device);
    return push_control(c, true);
}

int mmc_set_demag(mmc_ctx* c, int enabled, int updates_per_sweep)
{
    if (!c) return MMC_E_INVALID;
    if (updates_per_sweep != 1 && updates_per_sweep != 2) return fail(c, MMC_E_INVALID, "updates_per_sweep must be 1 or 2");
    DeviceGuard dg(c->device);
    if (c->demag_enabled && !enabled) {
        for (int q = 0; q < 3; ++q) cudaMemsetAsync(c->bd[q], 0, (size_t)(2 * c->g.H) * sizeof(float), c->stream);
        c->bd_version = 0;
    }
    c->demag_enabled = enabled ? 1 : 0; c->demag_updates = updates_per_sweep; c->dirty = true; c->args_version++;
    return MMC_OK;
}

int mmc_set_seed(mmc_ctx* c, uint64_t seed) { if (!c) return MMC_E_INVALID; c->seed = seed; c->args_version++; return MMC_OK; }

int mmc_set_sweep_counter(mmc_ctx* c, uint64_t sweep)
{
    if (!c) return MMC_E_INVALID;
    DeviceGuard dg(c->device);
    unsigned long long s = sweep;
    CU(c, cudaMemcpyAsync(&c->ctl->sweep, &s, sizeof(s), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return MMC_OK;
}

int mmc_set_m(mmc_ctx* c, const float* mx, const float* my, const float* mz)
{
    if (!c || !mx || !my || !mz) return fail(c, MMC_E_INVALID, "NULL pointer");
    DeviceGuard dg(c->device);
    const float* src[3] = { mx, my, mz };
    for (int q = 0; q < 3; ++q) {
        CU(c, cudaMemsetAsync(c->m[q], 0, (size_t)(2 * c->g.H) * sizeof(float), c->stream));
        int rc = launch_to_split(c->g, src[q], c->m[q], c->stream);
        if (rc) return fail(c, rc, "to_split launch failed");
    }
    c->m_set = true; c->state_version++;
    if (c->material_set && c->T_set) {
        int rc = ensure_setup(c); if (rc) return rc;
        return check_m(c);
    }
    c->m_needs_check = true;
    return MMC_OK;
}

int mmc_set_m_host(mmc_ctx* c, const float* mx, const float* my, const float* mz)
{
    if (!c || !mx || !my || !mz) return fail(c, MMC_E_INVALID, "NULL pointer");
    DeviceGuard dg(c->device);
    const size_t N = (size_t)c->g.nx * c->g.ny * c->g.nz;
    const float* src[3] = { mx, my, mz };
    for (int q = 0; q < 3; ++q) {                      // one staging buffer, reused in stream order
        CU(c, cudaMemcpyAsync(c->stage, src[q], N * sizeof(float), cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaMemsetAsync(c->m[q], 0, (size_t)(2 * c->g.H) * sizeof(float), c->stream));
        int rc = launch_to_split(c->g, c->stage, c->m[q], c->stream);
        if (rc) return fail(c, rc, "to_split launch failed");
    }
    c->m_set = true; c->state_version++;
    if (c->material_set && c->T_set) {
        int rc = ensure_setup(c); if (rc) return rc;
        return check_m(c);
    }
    c->m_needs_check = true;
    return MMC_OK;
}

int mmc_get_m_host(mmc_ctx* c, float* mx, float* my, float* mz)
{
    if (!c || !mx || !my || !mz) return fail(c, MMC_E_INVALID, "NULL pointer");
    DeviceGuard dg(c->device);
    const size_t N = (size_t)c->g.nx * c->g.ny * c->g.nz;
    float* dst[3] = { mx, my, mz };
    for (int q = 0; q < 3; ++q) {
        int rc = launch_from_split(c->g, c->m[q], c->stage, c->stream);
        if (rc) return fail(c, rc, "from_split launch failed");
        CU(c, cudaMemcpyAsync(dst[q], c->stage, N * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    }
    return MMC_OK;
}

int mmc_get_m(mmc_ctx* c, float* mx, float* my, float* mz)
{
    if (!c || !mx || !my || !mz) return fail(c, MMC_E_INVALID, "NULL pointer");
    DeviceGuard dg(c->device);
    float* dst[3] = { mx, my, mz };
    for (int q = 0; q < 3; ++q) { int rc = launch_from_split(c->g, c->m[q], dst[q], c->stream); if (rc) return fail(c, rc, "from_split launch failed"); }
    return MMC_OK;
}

// One iteration, enqueued on `st`: [demag] -> red -> [demag] -> black -> end of sweep.
static int enqueue_iteration(mmc_ctx* c, cudaStream_t st, PhaseTimer* timer, bool field_is_current)
{
    int rc;
    // the field is fully computed at the start of the iteration (skipped when bd[] already holds the
    // field of exactly this state, e.g. straight after a read-out) and frozen for the passes
    if (c->demag_enabled && !field_is_current) { rc = compute_demag(c, timer, st, true); if (rc) return rc; }
    c->state_version++;
    rc = launch_colour_pass(make_args(c, 0), c->features, false, st, &c->tma);
    if (rc) return fail(c, rc, "red pass launch failed");
    if (timer) timer->mark(PH_RED, st);
    if (c->demag_enabled && c->demag_updates == 2) { rc = compute_demag(c, timer, st, true); if (rc) return rc; }
    c->state_version++;
    // S11: on launch-bound meshes the last CTA of the black pass does the end-of-sweep bookkeeping itself (one launch less per
    // iteration: ~3 us of the ~22 us of BASELINE config 2); on large meshes the per-CTA fence + ticket costs more than the
    // one-thread launch it saves (config 4, 4096 CTAs: +6 us on the pass against a 3 us launch), so the separate kernel stays
    const bool fuse_end = (long long)c->g.nx * c->g.ny * c->g.nz <= (1ll << 20);
    SweepArgs black = make_args(c, 1);
    black.finish = fuse_end ? 1 : 0;
    rc = launch_colour_pass(black, c->features, false, st, &c->tma);
    if (rc) return fail(c, rc, "black pass launch failed");
    if (timer) timer->mark(PH_BLACK, st);
    if (!fuse_end) { rc = launch_end_sweep(c->ctl, st); if (rc) return fail(c, rc, "end_sweep launch failed"); }
    if (timer) timer->mark(PH_END, st);
    return MMC_OK;
}

constexpr int kGraphIters = 16;                       // iterations in the long graph

// Capture `iters` iterations into an executable graph.  Any failure switches graphs off for this ctx (plain launches go on).
static bool build_graph(mmc_ctx* c, int iters, mmc_ctx::IterGraph* g)
{
    if (g->exec) { cudaGraphExecDestroy(g->exec); g->exec = nullptr; }
    g->version = 0;
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { c->graphs_off = true; cudaGetLastError(); return false; }
    if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) { c->graphs_off = true; cudaGetLastError(); return false; }
    const uint64_t sv = c->state_version, bv = c->bd_version;
    int rc = MMC_OK;
    for (int it = 0; it < iters && rc == MMC_OK; ++it) rc = enqueue_iteration(c, c->cap_stream, nullptr, false);
    c->state_version = sv; c->bd_version = bv;        // nothing ran
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
    if (rc != MMC_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&g->exec, graph, 0) != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        g->exec = nullptr; c->graphs_off = true; cudaGetLastError();
        return false;
    }
    cudaGraphDestroy(graph);
    g->version = c->args_version;
    return true;
}

static int sweep_impl(mmc_ctx* c, int n_sweeps, PhaseTimer* timer)
{
    if (!c || n_sweeps < 0) return fail(c, MMC_E_INVALID, "n_sweeps >= 0 required");
    DeviceGuard dg(c->device);
    int rc = ready(c); if (rc) return rc;
    if (c->demag_enabled) { rc = ensure_demag(c); if (rc) return rc; }
    if (!timer && !c->demag_enabled && n_sweeps > 0) {            // small meshes: all iterations in one launch
        rc = launch_small_mesh_sweeps(make_args(c, 0), c->features, n_sweeps, c->stream);
        if (rc == MMC_OK) { c->state_version++; return MMC_OK; }
        if (rc != MMC_E_UNSUPPORTED) return fail(c, rc, "small-mesh launch failed");
    }
    if (timer) timer->mark(-1, c->stream);
    int left = n_sweeps;
    if (!timer && !c->graphs_off && left > 0) {
        // The first iteration after a change of settings runs as plain launches (it also loads the kernels and builds the demag
        // plan outside any capture); from then on whole iterations are replayed from graphs: 16 at a time, then one at a time.
        if (c->graph1.version != c->args_version) {
            rc = enqueue_iteration(c, c->stream, nullptr, c->bd_version == c->state_version); if (rc) return rc;
            --left;
            build_graph(c, 1, &c->graph1);
        }
        if (!c->graphs_off && left >= 2 * kGraphIters && c->graphN.version != c->args_version) build_graph(c, kGraphIters, &c->graphN);
        while (!c->graphs_off && left > 0) {
            const bool big = left >= kGraphIters && c->graphN.version == c->args_version && c->graphN.exec;
            if (!big && !(c->graph1.version == c->args_version && c->graph1.exec)) break;
            if (cudaGraphLaunch(big ? c->graphN.exec : c->graph1.exec, c->stream) != cudaSuccess) { c->graphs_off = true; cudaGetLastError(); break; }
            const int done = big ? kGraphIters : 1;
            left -= done; c->state_version += 2ull * done; c->bd_version = 0;
        }
    }
    for (; left > 0; --left) {
        rc = enqueue_iteration(c, c->stream, timer, !timer && c->bd_version == c->state_version);
        if (rc) return rc;
    }
    return MMC_OK;
}

int mmc_sweep(mmc_ctx* c, int n_sweeps) { return sweep_impl(c, n_sweeps, nullptr); }

int mmc_sweep_timed(mmc_ctx* c, int n_sweeps, double* phase_ms)
{
    if (!c || !phase_ms) return fail(c, MMC_E_INVALID, "NULL pointer");
    PhaseTimer t;
    int rc = sweep_impl(c, n_sweeps, &t);
    DeviceGuard dg(c->device);
    cudaStreamSynchronize(c->stream);
    for (int p = 0; p < PH_COUNT; ++p) phase_ms[p] = 0.0;
    for (size_t i = 1; i < t.events.size(); ++i) {
        float ms = 0.f;
        if (t.phase[i] >= 0 && cudaEventElapsedTime(&ms, (cudaEvent_t)t.events[i - 1], (cudaEvent_t)t.events[i]) == cudaSuccess)
            phase_ms[t.phase[i]] += (double)ms;
    }
    for (void* e : t.events) cudaEventDestroy((cudaEvent_t)e);
    if (rc == MMC_OK && t.failed) return fail(c, MMC_E_CUDA, "mmc_sweep_timed: a timing event could not be created or recorded");
    return rc;
}

int mmc_demag_field(mmc_ctx* c, float* bx, float* by, float* bz)
{
    if (!c) return MMC_E_INVALID;
    DeviceGuard dg(c->device);
    int rc = ready(c); if (rc) return rc;
    rc = compute_demag(c); if (rc) return rc;
    float* dst[3] = { bx, by, bz };
    for (int q = 0; q < 3; ++q)
        if (dst[q]) { rc = launch_from_split(c->g, c->bd[q], dst[q], c->stream); if (rc) return fail(c, rc, "from_split launch failed"); }
    if (!c->demag_enabled) {                     // keep the sweep's field term off
        for (int q = 0; q < 3; ++q) CU(c, cudaMemsetAsync(c->bd[q], 0, (size_t)(2 * c->g.H) * sizeof(float), c->stream));
        c->bd_version = 0;
    }
    return MMC_OK;
}

int mmc_get_observables(mmc_ctx* c, mmc_obs* out)
{
    if (!c || !out) return fail(c, MMC_E_INVALID, "NULL pointer");
    DeviceGuard dg(c->device);
    int rc = ready(c); if (rc) return rc;
    if (c->demag_enabled && c->bd_version != c->state_version) { rc = compute_demag(c); if (rc) return rc; }   // E_demag: field of the current state
    SweepArgs a = make_args(c, 0);
    if (!c->demag_enabled) a.bd[0] = a.bd[1] = a.bd[2] = nullptr;
    ObsParams op{};
    op.K1T_u = c->K1T_u; op.c0_u = c->c0_u;
    op.aex[0] = c->A0 * c->V / (c->dx * c->dx); op.aex[1] = c->A0 * c->V / (c->dy * c->dy); op.aex[2] = c->A0 * c->V / (c->dz * c->dz);
    op.D0V = c->D0 * c->V; op.inv_d[0] = 1.0 / c->dx; op.inv_d[1] = 1.0 / c->dy; op.kB = kBoltzmann;
    op.T_u = c->T_cell.empty() ? (float)c->T_uniform : (c->percell ? 1.f : c->T_cell[0]);
    if (!c->percell && !c->T_cell.empty()) {
        // uniform mode with a per-cell array means all active cells share one temperature: find it
        const long long N = (long long)c->g.nx * c->g.ny * c->g.nz;
        for (long long i = 0; i < N; ++i) {
            const int r = c->region_of_cell.empty() ? 0 : c->region_of_cell[i];
            if (c->regions[r].Ms0 > 0) { op.T_u = c->T_cell[i]; break; }
        }
    }
    rc = launch_observables(a, c->percell, op, c->d_obs, c->obs_scratch, c->obs_blocks, c->stream);
    if (rc) return fail(c, rc, "observables launch failed");
    CU(c, cudaMemcpyAsync(c->h_obs, c->d_obs, sizeof(ReadOut), cudaMemcpyDeviceToHost, c->stream));   // sums, control block, running sums
    CU(c, cudaStreamSynchronize(c->stream));
    const Observables ho = c->h_obs->obs; const Control hc = c->h_obs->ctl;
    long long fixed[4];
    for (int q = 0; q < 4; ++q) fixed[q] = (long long)c->h_obs->run_sums[q];
    std::memset(out, 0, sizeof(*out));
    const double na = ho.n_active > 0 ? (double)ho.n_active : 1.0;
    for (int q = 0; q < 3; ++q) out->mean_m[q] = ho.sum[q] / na;
    out->mean_len = ho.sum[3] / na;
    out->E_ex = ho.E[0]; out->E_an = ho.E[1]; out->E_zee = ho.E[2]; out->E_dmi = ho.E[3]; out->E_demag = ho.E[4]; out->E_long = ho.E[5];
    out->accepted = hc.accepted + hc.win_accepted; out->trials = hc.trials + hc.win_trials; out->sweeps_done = hc.sweep;
    out->cone_deg = hc.cone_deg; out->sigma_used = c->sigma_first;
    double rs[4] = { 0, 0, 0, 0 };
    for (int q = 0; q < 4; ++q) rs[q] = (double)fixed[q] / (double)kSumScale;
    out->run_sweeps = hc.run_sweeps;
    if (hc.run_sweeps > 0) {
        const double d = (double)hc.run_sweeps * na;
        for (int q = 0; q < 3; ++q) out->run_mean_m[q] = rs[q] / d;
        out->run_mean_len = rs[3] / d;
    }
    return MMC_OK;
}

int mmc_reset_counters(mmc_ctx* c)
{
    if (!c) return MMC_E_INVALID;
    DeviceGuard dg(c->device);
    Control h;
    CU(c, cudaMemcpyAsync(&h, c->ctl, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    // the read-out is accepted + win_accepted: zero it without disturbing the cone controller's 100-iteration window
    // (unsigned wrap-around: the window's counts are added back when it closes)
    h.accepted = 0ull - h.win_accepted; h.trials = 0ull - h.win_trials;
    CU(c, cudaMemcpyAsync(c->ctl, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return MMC_OK;
}

int mmc_reset_averages(mmc_ctx* c)
{
    if (!c) return MMC_E_INVALID;
    DeviceGuard dg(c->device);
    unsigned long long z = 0;
    CU(c, cudaMemsetAsync(c->run_sums, 0, 4 * sizeof(unsigned long long), c->stream));
    CU(c, cudaMemcpyAsync(&c->ctl->run_sweeps, &z, sizeof(z), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return MMC_OK;
}

int mmc_histogram(mmc_ctx* c, int kind, int nbins, double lo, double hi, uint64_t* counts, uint64_t* under_over)
{
    if (!c || !counts) return fail(c, MMC_E_INVALID, "NULL pointer");
    if ((kind != 0 && kind != 1) || nbins < 1 || nbins > 4096 || !(hi > lo) || !std::isfinite(lo) || !std::isfinite(hi))
        return fail(c, MMC_E_INVALID, "kind 0 or 1, 1 <= nbins <= 4096 and finite lo < hi required");
    DeviceGuard dg(c->device);
    int rc = ready(c); if (rc) return rc;
    double dir[3] = { 0.0, 0.0, 1.0 };
    if (kind == 1) {
        mmc_obs ob;
        rc = mmc_get_observables(c, &ob); if (rc) return rc;
        const double n = std::sqrt(ob.mean_m[0] * ob.mean_m[0] + ob.mean_m[1] * ob.mean_m[1] + ob.mean_m[2] * ob.mean_m[2]);
        if (!(n > 0)) return fail(c, MMC_E_INVALID, "the mean magnetisation vanishes: no mean direction");
        for (int q = 0; q < 3; ++q) dir[q] = ob.mean_m[q] / n;
    }
    unsigned long long* d = nullptr;
    CU(c, cudaMalloc(&d, (size_t)(nbins + 2) * sizeof(unsigned long long)));
    rc = launch_histogram(c->g, c->m, c->mask, kind, dir, nbins, lo, hi, d, c->stream);
    std::vector<unsigned long long> h((size_t)nbins + 2);
    cudaError_t e = rc ? cudaErrorUnknown : cudaMemcpyAsync(h.data(), d, h.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d);
    if (rc) return fail(c, rc, "histogram launch failed");
    if (e != cudaSuccess) return fail(c, MMC_E_CUDA, std::string("histogram: ") + cudaGetErrorString(e));
    for (int b = 0; b < nbins; ++b) counts[b] = h[(size_t)b];
    if (under_over) { under_over[0] = h[(size_t)nbins]; under_over[1] = h[(size_t)nbins + 1]; }
    return MMC_OK;
}

int mmc_relax(mmc_ctx* c, double ux, double uy, double uz, int chunk_sweeps, int min_chunks, int max_chunks, double threshold,
              mmc_relax_result* out)
{
    if (!c || !out) return fail(c, MMC_E_INVALID, "NULL pointer");
    const double un = std::sqrt(ux * ux + uy * uy + uz * uz);
    if (!(un > 0) || chunk_sweeps < 1 || min_chunks < 2 || max_chunks < min_chunks || !(threshold >= 0))
        return fail(c, MMC_E_INVALID, "direction != 0, chunk_sweeps >= 1, 2 <= min_chunks <= max_chunks, threshold >= 0 required");
    std::memset(out, 0, sizeof(*out));
    double prev = 0.0;
    for (int n = 1; n <= max_chunks; ++n) {
        int rc = mmc_reset_averages(c); if (rc) return rc;
        rc = mmc_sweep(c, chunk_sweeps); if (rc) return rc;
        mmc_obs ob;
        rc = mmc_get_observables(c, &ob); if (rc) return rc;
        const double par = (ob.run_mean_m[0] * ux + ob.run_mean_m[1] * uy + ob.run_mean_m[2] * uz) / un;
        out->chunks_done = n; out->sweeps += (uint64_t)chunk_sweeps;
        out->mean_par_prev = prev; out->mean_par_last = par;
        for (int q = 0; q < 3; ++q) out->mean_m[q] = ob.run_mean_m[q];
        out->mean_len = ob.run_mean_len;
        if (n >= min_chunks && std::fabs(par - prev) <= threshold) { out->converged = 1; break; }
        prev = par;
    }
    return MMC_OK;
}

int mmc_debug_pass(mmc_ctx* c, int colour, float* dm, float* dF_terms, float* margin, uint8_t* accepted)
{
    if (!c || (colour != 0 && colour != 1)) return fail(c, MMC_E_INVALID, "colour must be 0 or 1");
    DeviceGuard dg(c->device);
    int rc = ready(c); if (rc) return rc;
    SweepArgs a = make_args(c, colour);
    a.run_sums = nullptr;
    a.dbg_dm = dm; a.dbg_terms = dF_terms; a.dbg_margin = margin; a.dbg_acc = accepted;
    rc = launch_colour_pass(a, c->features, true, c->stream);
    c->state_version++;
    if (rc) return fail(c, rc, "debug pass launch failed");
    return MMC_OK;
}

int mmc_thermal(double T, double Tc, double mu_atom, double V, double Ms0, double* out6)
{
    if (!out6) return MMC_E_INVALID;
    ThermalCoef t;
    int rc = thermal_coefficients(T, Tc, mu_atom, V, Ms0, &t);
    if (rc) return rc;
    out6[0] = t.me; out6[1] = t.chi; out6[2] = t.c2; out6[3] = t.c4; out6[4] = t.sigma13; out6[5] = t.mu2;
    return MMC_OK;
}

int mmc_demag_tensor_at(double dx, double dy, double dz, int ox, int oy, int oz, double* out6)
{
    if (!out6) return MMC_E_INVALID;
    return demag_tensor_at(dx, dy, dz, ox, oy, oz, kNearRadius, out6);
}

const char* mmc_strerror(int code)
{
    switch (code) {
        case MMC_OK: return "ok";
        case MMC_E_INVALID: return "invalid argument";
        case MMC_E_ZERO_LENGTH: return "zero-length magnetisation in a non-empty cell";
        case MMC_E_CUDA: return "CUDA error";
        case MMC_E_NOMEM: return "out of memory";
        case MMC_E_UNSUPPORTED: return "unsupported configuration";
        case MMC_E_STATE: return "call order: material, temperature and m must be set first";
        case MMC_E_TOO_LARGE: return "more cells than the static scratch array serves (MMC_STATIC_MAX_CELLS = 16777216)";
        default: return "unknown error";
    }
}

const char* mmc_last_error(const mmc_ctx* c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"
