// bb_api.cu -- C ABI of libbiobeam_b200.so (include/bb.h): argument checks, plan cache
// (twiddle tables, propagator tables, workspace), launch sequencing.  All arithmetic of the
// method runs in the kernels of bb_kernels.cuh / bb_aux_kernels.cuh.
#include "../../include/bb.h"
#include "bb_launch.h"
#include "bb_aux_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

extern char **environ;

namespace {

using bb::KParams;
typedef float2 cf;

thread_local std::string g_err;
std::mutex g_mu;
unsigned long long g_launches = 0;
long long *g_trace = nullptr;      // bb_probe_trace
int g_trace_phases = 0;
int g_trace_dev = -1;
char g_last_kernel[96] = "";      // bb_last_kernel

int fail(int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define BB_CUDA(call)                                                                         \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(e_ == cudaErrorMemoryAllocation ? BB_ERR_OOM : BB_ERR_CUDA,           \
                        "%s failed: %s", #call, cudaGetErrorString(e_));                      \
    } while (0)

const double kTwoPi = 6.283185307179586476925286766559;

int log2_exact(int n) {
    if (n <= 0 || (n & (n - 1))) return -1;
    int l = 0;
    while ((1 << l) < n) ++l;
    return l;
}

// ------------------------------------------------------------------------------------------
// Plan: everything cached for one (device, Nx, Ny).
// ------------------------------------------------------------------------------------------
struct TableKey {
    float dx, dz, lambda, nref;
    int perm;                      // column order: 1 natural, P = kx-class-major (16-point-thread kernel)
    bool operator==(const TableKey &o) const {
        return memcmp(this, &o, sizeof(TableKey)) == 0;
    }
};
struct TableEntry { TableKey key; cf *ptr; unsigned long long last_use; };

struct Plan {
    int device, Nx, Ny;
    cf *twx = nullptr, *twy = nullptr;
    cf *tw256 = nullptr, *twcx = nullptr, *twcy = nullptr;   // 16-point-thread kernel tables
    bool k16 = false;              // that kernel is available for this shape
    bool k8 = false;               // 8-point-thread kernel available for this shape
    bool k32 = false;              // 32-point-thread kernel (all shapes up to 1024; transform programs)
    bool force_k8 = false;         // BB_USE_K8=1 when the plan was made
    int kc_cs = 0;                 // cluster kernel (grids up to 256^2): CTAs per cluster, 0 = not available
    int kc_mode = 1;               // ... exchange: 1 bulk copies counted on mbarriers, 0 remote stores + cluster barriers (BB_KC_MODE)
    int kc_pt = 8;                 // ... points per thread: 16 on 256 x 256 (BB_KC_PT=8: the 8-point form there too)
    bool kc_force = false;         // BB_KC_FORCE=1: use it on 256 x 256 as well
    // diagnostic switches, read once when the plan is made (bb_shutdown + a new call re-reads them)
    bool env_notma = false, env_noprune = false;
    int env_cw = 0;                // BB_K16_CW: 4 or 8, 0 = automatic
    // pupil of the last bb_multiplex_* call on this grid (pixel count and bounding box: an O(Nx Ny) host loop)
    struct Pupil { float dx = 0.f, lambda = 0.f, na_in = -1.f, na = -1.f; long long count = 0; int Fx = 0, Wx = 0, Fy = 0, Wy = 0; } pupil;
    unsigned *bar = nullptr;
    int *status = nullptr;
    std::vector<TableEntry> tables;
    size_t table_capacity = 0;
    const cf **d_htab = nullptr;   // per-step arrays
    float *d_phase = nullptr;
    int *d_fmax = nullptr;         // per step: largest live |kx bin| (16-point-thread kernel)
    int cw4 = 0;                   // column tiles of 4 columns for the propagation being enqueued
    int step_cap = 0;
    int grid = 0;                  // persistent grid size (<= SM count)
    int run_grid = 0;              // grid of the propagation being enqueued (small grids: one CTA per live column tile)
    int sm_count = 0;
    unsigned long long tick = 0;
};

void destroy_plan(Plan *p) {
    for (void *q : {(void *)p->twx, (void *)p->twy, (void *)p->tw256, (void *)p->twcx, (void *)p->twcy, (void *)p->bar,
                    (void *)p->status, (void *)p->d_htab, (void *)p->d_phase, (void *)p->d_fmax})
        if (q) cudaFree(q);
    for (TableEntry &e : p->tables) cudaFree(e.ptr);
    delete p;
}

std::vector<Plan *> g_plans;
struct Workspace { void *ptr = nullptr; size_t bytes = 0; };
// Everything the library allocates outside a plan belongs to ONE device: workspaces of the host-buffer
// entry point and of the helpers, its copy / compute streams and their events (created once, reused).
struct DeviceCtx {
    Workspace field, dn, I, misc;
    cudaStream_t s_in = nullptr, s_run = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> events;
};
std::map<int, DeviceCtx> g_ctx;
DeviceCtx &device_ctx() {
    int dev = 0;
    cudaGetDevice(&dev);
    return g_ctx[dev];
}

int check_arch(int *device_out, int *sm_count) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(BB_ERR_CUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
    int major = 0, sms = 0;
    BB_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    BB_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10)
        return fail(BB_ERR_ARCH, "device %d has compute capability %d.x; this library is sm_100a only", dev, major);
    *device_out = dev;
    *sm_count = sms;
    return BB_OK;
}

std::vector<cf> make_twiddles(int N) {
    // tw[k1*T + t] = exp(-2 pi i k1 t / N), k1 < 32, t < T = N/32, from double
    int T = N / 32;
    std::vector<cf> tw((size_t)32 * T);
    for (int k1 = 0; k1 < 32; ++k1)
        for (int t = 0; t < T; ++t) {
            double ph = -kTwoPi * (double)((long long)k1 * t) / (double)N;
            tw[(size_t)k1 * T + t] = make_float2((float)cos(ph), (float)sin(ph));
        }
    return tw;
}

size_t table_budget_bytes() {
    const char *e = getenv("BB_TABLE_CACHE_MB");
    size_t mb = e ? (size_t)atoll(e) : 1024;
    if (mb < 16) mb = 16;
    return mb << 20;
}

// The diagnostic switches the library reads from the environment when it makes a plan.  A BB_* variable that is
// not one of them is a spelling mistake that would otherwise be ignored without a word: the call fails instead.
const char *const kEnvSwitches[] = {"BB_TABLE_CACHE_MB", "BB_DISABLE_K16", "BB_DISABLE_K8", "BB_USE_K8", "BB_DISABLE_KC",
                                    "BB_KC_MODE", "BB_KC_PT", "BB_KC_FORCE", "BB_KC_CS", "BB_K16_NOTMA", "BB_K16_NOPRUNE",
                                    "BB_K16_CW", "BB_GRID"};
int check_env_switches() {
    for (char **e = environ; e && *e; ++e) {
        if (strncmp(*e, "BB_", 3) != 0) continue;
        const char *eq = strchr(*e, '=');
        const size_t n = eq ? (size_t)(eq - *e) : strlen(*e);
        bool known = false;
        for (const char *k : kEnvSwitches) known = known || (strlen(k) == n && strncmp(k, *e, n) == 0);
        if (!known) return fail(BB_ERR_INVALID_ARG, "unknown environment switch %.*s (the library knows BB_TABLE_CACHE_MB, "
                                "BB_DISABLE_K16/K8/KC, BB_USE_K8, BB_KC_MODE/PT/FORCE/CS, BB_K16_NOTMA/NOPRUNE/CW, BB_GRID)",
                                (int)n, *e);
    }
    return BB_OK;
}

int get_plan(int Nx, int Ny, Plan **out) {
    int dev, sms;
    int rc = check_arch(&dev, &sms);
    if (rc) return rc;
    for (Plan *p : g_plans)
        if (p->device == dev && p->Nx == Nx && p->Ny == Ny) { *out = p; return BB_OK; }
    rc = check_env_switches();
    if (rc) return rc;
    Plan *p = new Plan();
    struct Guard { Plan *p; ~Guard() { if (p) destroy_plan(p); } } guard{p};   // every early return releases what was allocated
    p->device = dev; p->Nx = Nx; p->Ny = Ny; p->sm_count = sms;
    if (Nx <= 1024 && Ny <= 1024) {
        std::vector<cf> tx = make_twiddles(Nx), ty = make_twiddles(Ny);
        BB_CUDA(cudaMalloc(&p->twx, tx.size() * sizeof(cf)));
        BB_CUDA(cudaMalloc(&p->twy, ty.size() * sizeof(cf)));
        BB_CUDA(cudaMemcpy(p->twx, tx.data(), tx.size() * sizeof(cf), cudaMemcpyHostToDevice));
        BB_CUDA(cudaMemcpy(p->twy, ty.data(), ty.size() * sizeof(cf), cudaMemcpyHostToDevice));
    }
    BB_CUDA(cudaMalloc(&p->bar, 256));
    BB_CUDA(cudaMalloc(&p->status, 256));
    BB_CUDA(cudaMemset(p->bar, 0, 256));
    BB_CUDA(cudaMemset(p->status, 0, 256));
    const bool want16 = bb::kernel16_supports(Nx, Ny) && !getenv("BB_DISABLE_K16");
    const bool want8 = bb::kernel8_supports(Nx, Ny) && !getenv("BB_DISABLE_K8");
    if (want16 || want8) {
        // sub-line twiddles exp(-2 pi i k1 t / 256) and class twiddles exp(-2 pi i c q / N), c = 1..P-1, q < 256
        std::vector<cf> t256(256);
        for (int k1 = 0; k1 < 16; ++k1)
            for (int t = 0; t < 16; ++t) {
                double ph = -kTwoPi * (double)(k1 * t) / 256.0;
                t256[(size_t)k1 * 16 + t] = make_float2((float)cos(ph), (float)sin(ph));
            }
        auto class_tw = [](int N) {
            int P = N / 256;
            std::vector<cf> w((size_t)std::max(1, (P - 1) * 256));
            for (int c = 1; c < P; ++c)
                for (int q = 0; q < 256; ++q) {
                    double ph = -kTwoPi * (double)(c * q) / (double)N;
                    w[(size_t)(c - 1) * 256 + q] = make_float2((float)cos(ph), (float)sin(ph));
                }
            return w;
        };
        std::vector<cf> cx = class_tw(Nx), cy = class_tw(Ny);
        BB_CUDA(cudaMalloc(&p->tw256, t256.size() * sizeof(cf)));
        BB_CUDA(cudaMalloc(&p->twcx, cx.size() * sizeof(cf)));
        BB_CUDA(cudaMalloc(&p->twcy, cy.size() * sizeof(cf)));
        BB_CUDA(cudaMemcpy(p->tw256, t256.data(), t256.size() * sizeof(cf), cudaMemcpyHostToDevice));
        BB_CUDA(cudaMemcpy(p->twcx, cx.data(), cx.size() * sizeof(cf), cudaMemcpyHostToDevice));
        BB_CUDA(cudaMemcpy(p->twcy, cy.data(), cy.size() * sizeof(cf), cudaMemcpyHostToDevice));
        if (want16) {
            int rc16 = bb::kernel16_prepare(Nx, Ny);
            if (rc16 != 0) { return fail(BB_ERR_CUDA, "kernel16_prepare failed: %s", cudaGetErrorString((cudaError_t)rc16)); }
            if (bb::kernel16_blocks_per_sm(Nx, Ny) < 1) { return fail(BB_ERR_CUDA, "16-point BPM kernel does not fit on an SM"); }
            p->k16 = true;
        }
        if (want8) {
            int rc8 = bb::kernel8_prepare(Nx, Ny);
            if (rc8 != 0) { return fail(BB_ERR_CUDA, "kernel8_prepare failed: %s", cudaGetErrorString((cudaError_t)rc8)); }
            if (bb::kernel8_blocks_per_sm(Nx, Ny) < 1) { return fail(BB_ERR_CUDA, "8-point BPM kernel does not fit on an SM"); }
            p->k8 = true;
            p->force_k8 = getenv("BB_USE_K8") != nullptr;
        }
    }
    size_t tb = (size_t)Nx * Ny * sizeof(cf);
    p->table_capacity = std::max<size_t>(2, std::min<size_t>(4096, table_budget_bytes() / tb));
    if (Nx <= 1024 && Ny <= 1024) {
        rc = bb::kernel_prepare(Nx, Ny);
        if (rc != 0) { return fail(BB_ERR_CUDA, "kernel_prepare failed: %s", cudaGetErrorString((cudaError_t)rc)); }
        int per_sm = bb::kernel_blocks_per_sm(Nx, Ny);
        if (per_sm < 1) { return fail(BB_ERR_CUDA, "BPM kernel does not fit on an SM"); }
        p->k32 = true;
    }
    if (!p->k32 && !p->k8) { return fail(BB_ERR_UNSUPPORTED_SHAPE, "no kernel for Nx = %d, Ny = %d", Nx, Ny); }
    if (bb::kernelc_supports(Nx, Ny) && !getenv("BB_DISABLE_KC") && !getenv("BB_USE_K8")) {
        // the largest cluster the device schedules: 16 CTAs (non-portable size) halve the per-CTA share of the exchange
        p->kc_mode = getenv("BB_KC_MODE") ? (atoi(getenv("BB_KC_MODE")) != 0) : 1;
        p->kc_pt = Nx == 256 && Ny == 256 && !(getenv("BB_KC_PT") && atoi(getenv("BB_KC_PT")) == 8) ? 16 : 8;
        p->kc_force = getenv("BB_KC_FORCE") != nullptr;
        const int want = getenv("BB_KC_CS") ? atoi(getenv("BB_KC_CS")) : 0;
        for (int cs : {16, 8}) {
            if (want && cs != want) continue;
            if (bb::kernelc_prepare(Nx, Ny, cs, p->kc_mode, p->kc_pt) != 0) { (void)cudaGetLastError(); continue; }
            if (bb::kernelc_max_clusters(Nx, Ny, cs, p->kc_mode, p->kc_pt) >= 1) { p->kc_cs = cs; break; }
        }
    }
    p->grid = sms;
    p->env_notma = getenv("BB_K16_NOTMA") != nullptr;
    p->env_noprune = getenv("BB_K16_NOPRUNE") != nullptr;
    p->env_cw = getenv("BB_K16_CW") ? atoi(getenv("BB_K16_CW")) : 0;
    if (getenv("BB_GRID")) p->grid = std::max(1, std::min(sms, atoi(getenv("BB_GRID"))));   // diagnostic: persistent grid size
    guard.p = nullptr;
    g_plans.push_back(p);
    *out = p;
    return BB_OK;
}

int ensure_steps(Plan *p, int Nz) {
    if (Nz <= p->step_cap) return BB_OK;
    if (p->d_htab) { cudaFree((void *)p->d_htab); cudaFree(p->d_phase); cudaFree(p->d_fmax); p->d_htab = nullptr; p->d_phase = nullptr; p->d_fmax = nullptr; }
    int cap = std::max(Nz, 1024);
    BB_CUDA(cudaMalloc((void **)&p->d_htab, (size_t)cap * sizeof(cf *)));
    BB_CUDA(cudaMalloc(&p->d_phase, (size_t)cap * sizeof(float)));
    BB_CUDA(cudaMalloc(&p->d_fmax, (size_t)cap * sizeof(int)));
    p->step_cap = cap;
    return BB_OK;
}

int build_table(Plan *p, const TableKey &k, cf *dst, cudaStream_t s) {
    double k0 = kTwoPi / (double)k.lambda;
    double kk = k0 * (double)k.nref;
    dim3 block(128), grid((p->Nx + 127) / 128, p->Ny);
    bb::propagator_table_kernel<<<grid, block, 0, s>>>(dst, p->Nx, p->Ny, (double)k.dx, (double)k.dz, kk,
                                                       1.0 / ((double)p->Nx * (double)p->Ny), k.perm);
    ++g_launches;
    BB_CUDA(cudaGetLastError());
    return BB_OK;
}

// Largest |DFT bin| f of an N-point axis with pitch dx for which the propagator of wavenumber k can be
// non-zero (bb.h step 2: s = k^2 - kx^2 - ky^2 > 0 needs kx^2 < k^2).  Conservative: a bin within
// 1e-9 of the cut counts as live (a live column that is in fact all zero is only computed in vain).
int live_fmax(int N, double dx, double k) {
    const double lim = k * k * (1.0 + 1e-9);
    int f = (int)std::floor(k * (double)N * dx / kTwoPi);
    f = std::max(0, std::min(f, N / 2));
    auto kx2 = [&](int g) { double kx = kTwoPi * (double)g / ((double)N * dx); return kx * kx; };
    while (f < N / 2 && kx2(f + 1) < lim) ++f;
    while (f > 0 && !(kx2(f) < lim)) --f;
    return f;
}

// Number of live column tiles of width cw (the host copy of bb::LiveCols::total, bb_kernels16.cuh).
int live_tiles(int N, int F, int cw) {
    const int P = N / 256, L = 256, ntc = L / cw;
    int n = 0;
    for (int c = 0; c < P; ++c) {
        int lo_cols = F >= c ? (F - c) / P + 1 : 0;
        lo_cols = std::min(lo_cols, L);
        int hs = std::min((N - F - c + P - 1) / P, L);
        int a = (lo_cols + cw - 1) / cw, b = ntc - hs / cw;
        if (a + b >= ntc) { a = ntc; b = 0; }
        n += a + b;
    }
    return n;
}

// Tile width of the column phase for a whole propagation (it must not change between the launches of
// one propagation): 4 columns when the (tile, field) units then still fit one per SM, else 8.
bool use_k16(const Plan *p, int B);

void choose_tile_width(Plan *p, int B, int Nz, float dx, float lambda, float n0, const float *nref) {
    p->cw4 = 0;
    p->run_grid = p->grid;
    if (!p->k16 && !p->k8) return;
    if (p->Ny > 1024) { p->cw4 = 1; return; }          // a tile of 8 columns x 2048 rows exceeds one team
    double k0 = kTwoPi / (double)lambda;
    int F = 0;
    for (int j = 0; j < Nz; ++j) F = std::max(F, live_fmax(p->Nx, (double)dx, k0 * (double)(nref ? nref[j] : n0)));
    if (p->env_cw) { p->cw4 = p->env_cw == 4; return; }
    p->cw4 = live_tiles(p->Nx, F, 4) * B <= p->grid;
    // A small single field leaves most SMs without a column tile: a grid of one CTA per live tile has the
    // same critical path (one tile per CTA, a few rows per CTA in parallel teams) and a cheaper grid barrier
    // (256^2: 8.8 -> 8.0 us per step).  Only when it at least halves the grid (144 CTAs instead of 148 lose at 1024^2).
    if (B == 1 && use_k16(p, B)) {
        const int t = live_tiles(p->Nx, F, p->cw4 ? 4 : 8);
        if (t >= 1 && 2 * t <= p->grid) p->run_grid = t;
    }
}

constexpr int kTableCacheFull = -1;   // internal: every cached table belongs to the launch being assembled

// Returns the cached table for `k`, building it on `s` if needed.  Entries used at
// tick >= protect_tick are never recycled (they belong to the launch being assembled).
int get_table(Plan *p, const TableKey &k, cudaStream_t s, unsigned long long protect_tick, cf **out) {
    for (TableEntry &e : p->tables)
        if (e.key == k) { e.last_use = p->tick; *out = e.ptr; return BB_OK; }
    TableEntry *slot = nullptr;
    if (p->tables.size() < p->table_capacity) {
        TableEntry e;
        e.ptr = nullptr;
        cudaError_t ce = cudaMalloc(&e.ptr, (size_t)p->Nx * p->Ny * sizeof(cf));
        if (ce == cudaSuccess) { p->tables.push_back(e); slot = &p->tables.back(); }
        else (void)cudaGetLastError();
    }
    if (!slot) {
        for (TableEntry &e : p->tables)
            if (e.last_use < protect_tick && (!slot || e.last_use < slot->last_use)) slot = &e;
        if (!slot) return kTableCacheFull;
    }
    slot->key = TableKey{0.f, 0.f, 0.f, -1.f, 0};            // no table until the build has been enqueued
    int rc = build_table(p, k, slot->ptr, s);
    if (rc) return rc;
    slot->key = k;
    slot->last_use = p->tick;
    *out = slot->ptr;
    return BB_OK;
}

// Supported grids: powers of two in [32, 2048]; 2048-point lines exist only in the 8-point-thread
// kernel, which needs both sides >= 256.
bool shape_ok(int Nx, int Ny) {
    const int lx = log2_exact(Nx), ly = log2_exact(Ny);
    if (lx < 5 || lx > 11 || ly < 5 || ly > 11) return false;
    if ((lx == 11 || ly == 11) && (lx < 8 || ly < 8)) return false;
    return true;
}

int validate_common(const void *field, const float *dn, int Nx, int Ny, int Nz, float dx, float dz,
                    float lambda, float n0, const bb_opts *opts, int *B, unsigned *flags) {
    if (!field) return fail(BB_ERR_INVALID_ARG, "field is NULL");
    const bool homogeneous = opts && (opts->flags & BB_HOMOGENEOUS);
    if (!dn && !homogeneous) return fail(BB_ERR_INVALID_ARG, "dn_volume is NULL (only BB_HOMOGENEOUS runs without one)");
    if (Nz < 1) return fail(BB_ERR_INVALID_ARG, "Nz = %d must be >= 1", Nz);
    if (!(dx > 0.f) || !(dz > 0.f) || !(lambda > 0.f) || !(n0 > 0.f) || !std::isfinite(dx) ||
        !std::isfinite(dz) || !std::isfinite(lambda) || !std::isfinite(n0))
        return fail(BB_ERR_INVALID_ARG, "dx, dz, lambda, n0 must be positive and finite");
    if (!shape_ok(Nx, Ny))
        return fail(BB_ERR_UNSUPPORTED_SHAPE, "Nx = %d, Ny = %d: both must be powers of two in [32, 2048], and both >= 256 if one is 2048", Nx, Ny);
    *B = 1;
    *flags = 0;
    if (opts) {
        if (opts->struct_size != (int)sizeof(bb_opts))
            return fail(BB_ERR_INVALID_ARG, "bb_opts.struct_size = %d, expected %d", opts->struct_size, (int)sizeof(bb_opts));
        if (opts->batch < 1) return fail(BB_ERR_INVALID_ARG, "batch = %d must be >= 1", opts->batch);
        if (opts->flags & ~(BB_ACCUMULATE | BB_INTENSITY_PER_FIELD | BB_LAUNCH_PER_PHASE | BB_BACKWARD | BB_HOMOGENEOUS))
            return fail(BB_ERR_INVALID_ARG, "unknown flag bits 0x%x", opts->flags);
        if (homogeneous && opts->nref)
            return fail(BB_ERR_INVALID_ARG, "BB_HOMOGENEOUS propagates in the medium n0: nref must be NULL");
        if (opts->nref)
            for (int j = 0; j < Nz; ++j)
                if (!(opts->nref[j] > 0.f) || !std::isfinite(opts->nref[j]))
                    return fail(BB_ERR_INVALID_ARG, "nref[%d] must be positive and finite", j);
        *B = opts->batch;
        *flags = opts->flags;
    }
    return BB_OK;
}

// cuTensorMapEncodeTiled through the runtime (no link against libcuda): the descriptor the TMA unit
// uses to fetch column tiles of the field (bb_kernels16.cuh).
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
        else
            (void)cudaGetLastError();
    }
    return fn;
}
// fields [B][Ny][Nx] of 8-byte elements as (column, y mod PY, y div PY, field); box = (cw, 1, 256, 1)
bool make_field_tmap(CUtensorMap *tm, void *field, int Nx, int Ny, int B, int cw) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const int PY = Ny / 256;
    cuuint64_t dims[4] = {(cuuint64_t)Nx, (cuuint64_t)PY, 256, (cuuint64_t)B};
    cuuint64_t strides[3] = {(cuuint64_t)Nx * 8, (cuuint64_t)PY * Nx * 8, (cuuint64_t)Nx * Ny * 8};
    cuuint32_t box[4] = {(cuuint32_t)cw, 1, 256, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, field, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              // L2 promotion: NONE; 64 / 128 / 256 B measured on C4 (round 3): 13.626 / 13.630 / 13.642 ms against 13.627 -- no effect
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The 16-point-thread kernel serves single fields on 256/512/1024 grids; everything else (batches,
// other shapes, the generic transform programs) runs on the 32-point-thread kernel.
// The 16-point-thread kernel is faster wherever both apply (profiles/r02_k8_kernel.md); the 8-point-thread one serves the
// transform programs of 2048-point lines (run_program) and is a diagnostic alternative for propagations (BB_USE_K8=1).
bool use_k8(const Plan *p, int B) {
    if (!p->k8) return false;
    if (p->k16 && !p->force_k8) return false;
    const int rows = (p->Ny + p->grid - 1) / p->grid;
    return B == 1 || (long long)rows * p->Nx <= 8192;
}
bool use_k16(const Plan *p, int B) {
    if (!p->k16 || use_k8(p, B)) return false;
    // the batch variant shares one buffer of screen factors among the teams: all rows of a CTA must fit
    const int rows = (p->Ny + p->grid - 1) / p->grid;
    return B == 1 || (long long)rows * p->Nx <= 8192;
}

// The cluster kernel (bb_kernelsc.cuh: one cluster per field, the field in distributed shared memory) takes every
// grid with a 128-point side that it supports: 2.5 - 5 x faster than the grid kernels there, single fields and
// batches (profiles/r02_cluster_kernel.md).  On 256 x 256 it only ties with the 16-point-thread grid kernel for a
// single field (both 7.8 us per step: the exchange is bound by the 16 CTAs' distributed-shared-memory bandwidth) and
// loses for batches of 16 and more, so it is not used there unless BB_KC_FORCE=1 (tests, measurements).
bool use_kc(const Plan *p, int B) {
    (void)B;
    if (p->kc_cs == 0) return false;
    return p->kc_force || p->Nx == 128 || p->Ny == 128;
}

int batch_warps(int B) {
    int bw = 1;
    while (bw < B && bw < bb::kWarps) bw <<= 1;
    return bw;
}

// Enqueue steps [j0, j1) of a propagation of Nz_total steps.  dn / inten point at slice j0.
// Tables and per-step arrays for [j0, j1) must already be in place.
int launch_steps(Plan *p, cf *field, const float *dn, float *inten, long long inten_bstride, int B,
                 int Nz_total, int j0, int j1, float phase_b, unsigned flags, cudaStream_t s) {
    KParams P;
    memset(&P, 0, sizeof P);
    P.field = field; P.inten = inten; P.inten_bstride = inten_bstride;
    P.dn = dn ? dn : reinterpret_cast<const float *>(field);   // BB_HOMOGENEOUS: never read, only tells the slices apart
    P.htab = p->d_htab; P.phase_a = p->d_phase; P.phase_b = phase_b;
    P.Nx = p->Nx; P.Ny = p->Ny; P.B = B; P.BW = batch_warps(B);
    P.Nz_total = Nz_total; P.j_base = j0;
    P.mode = 0;
    P.twx = p->twx; P.twy = p->twy; P.bar = p->bar; P.status = p->status;
    P.tw256 = p->tw256; P.twcx = p->twcx; P.twcy = p->twcy;
    P.fmax = p->d_fmax; P.cw4 = p->cw4;
    P.flags = flags & 3u;
    P.backward = (flags & BB_BACKWARD) ? 1 : 0;
    P.noscreen = (flags & BB_HOMOGENEOUS) ? 1 : 0;
    const bool kc = use_kc(p, B);
    const bool k8 = !kc && use_k8(p, B), k16 = !kc && use_k16(p, B);
    if (!kc && !k8 && !k16 && !p->k32) return fail(BB_ERR_UNSUPPORTED_SHAPE, "no kernel for Nx = %d, Ny = %d, batch = %d", p->Nx, p->Ny, B);
    if (k16 || k8) P.use_tma = !p->env_notma && make_field_tmap(&P.tmap, field, p->Nx, p->Ny, B, p->cw4 ? 4 : 8) ? 1 : 0;
    // The trace buffer holds [phases][SM count][6] records.  The grid kernels never launch more CTAs than SMs; the cluster
    // kernel launches kc_cs * B of them, which fits for a single field only (kc_cs <= 16), so batches there are not traced.
    if (g_trace && g_trace_dev == p->device && ((kc && B == 1) || k16 || k8) && 2 * Nz_total + 1 <= g_trace_phases) { P.trace = g_trace; P.trace_p0 = 0; }
    snprintf(g_last_kernel, sizeof g_last_kernel, k8 ? "bb::bpm8_kernel<%d,%d,%d,%s>" : k16 ? "bb::bpm16_kernel<%d,%d,%d,%s>" : "bb::bpm_kernel<%d,%d,%d>",
             k8 || k16 ? p->Nx / 256 : p->Nx / 32, k8 || k16 ? p->Ny / 256 : p->Ny / 32, k8 || k16 ? (p->cw4 ? 4 : 8) : 8,
             B > 1 ? "true" : "false");
    if (kc) snprintf(g_last_kernel, sizeof g_last_kernel, "bb::bpmc_kernel<%d,%d,%d,%d,%d>", p->Nx, p->Ny, p->kc_cs, p->kc_mode, p->kc_pt);
    auto launch = [&](bool coop) {
        return kc ? bb::kernelc_launch(p->Nx, p->Ny, p->kc_cs, p->kc_mode, p->kc_pt, P, B, s)
             : k8 ? bb::kernel8_launch(p->Nx, p->Ny, P, p->grid, coop, s)
                  : k16 ? bb::kernel16_launch(p->Nx, p->Ny, P, p->run_grid > 0 ? p->run_grid : p->grid, coop, s)
                        : bb::kernel_launch(p->Nx, p->Ny, P, p->grid, coop, s);
    };
    // steps [j0, j1): forward = column phases j0 .. j1-1 and the row phases after them (plus row phase 0);
    // backward = row / column phases Nz-j1 .. Nz-1-j0 in that order (plus the closing row phase Nz)
    int p0 = (j0 == 0) ? 0 : 2 * j0 + 1, p1 = 2 * j1 + 1;
    if (kc && B > 1 && inten && !(flags & BB_INTENSITY_PER_FIELD) && !(flags & BB_ACCUMULATE))
        BB_CUDA(cudaMemsetAsync(inten, 0, (size_t)(j1 - j0) * p->Nx * p->Ny * sizeof(float), s));   // the clusters add into it
    if (flags & BB_BACKWARD) { p0 = 2 * (Nz_total - j1); p1 = 2 * (Nz_total - j0) + (j0 == 0 ? 1 : 0); }
    if (flags & BB_LAUNCH_PER_PHASE) {
        for (int ph = p0; ph < p1; ++ph) {
            P.p0 = ph; P.p1 = ph + 1;
            cudaError_t e = launch(false);
            ++g_launches;
            if (e != cudaSuccess) return fail(BB_ERR_CUDA, "phase launch failed: %s", cudaGetErrorString(e));
        }
    } else {
        P.p0 = p0; P.p1 = p1;
        BB_CUDA(cudaMemsetAsync(p->bar, 0, sizeof(unsigned), s));
        cudaError_t e = launch(true);
        ++g_launches;
        if (e != cudaSuccess) return fail(BB_ERR_CUDA, "cooperative launch failed: %s", cudaGetErrorString(e));
    }
    return BB_OK;
}

// Per-step tables and phase offsets for the steps at positions [i0, *i_done) of the processing order
// (forward: step j = i; backward: j = Nz - 1 - i): the longest run whose distinct propagator tables
// fit the cache together (normally all of it).  Backward steps use the conjugate factors, i.e. the
// table and the phase offset of -dz.
int prepare_steps(Plan *p, int B, int Nz, int i0, float dx, float dz, float lambda, float n0, const float *nref,
                  unsigned flags, cudaStream_t s, std::vector<const cf *> &h_tab, std::vector<float> &h_phase, int *i_done) {
    std::vector<int> h_fmax(Nz);
    const bool backward = (flags & BB_BACKWARD) != 0;
    const float dzs = backward ? -dz : dz;
    double k0 = kTwoPi / (double)lambda;
    unsigned long long protect = ++p->tick;
    const cf *last_ptr = nullptr;
    float last_nref = 0.f;
    const bool noprune = p->env_noprune;
    int i = i0;
    for (; i < Nz; ++i) {
        const int j = backward ? Nz - 1 - i : i;
        float nr = nref ? nref[j] : n0;
        if (!(last_ptr && nr == last_nref)) {
            TableKey key = {dx, dzs, lambda, nr, (use_k16(p, B) || use_k8(p, B)) ? p->Nx / 256 : 1};
            cf *ptr = nullptr;
            int rc = get_table(p, key, s, protect, &ptr);
            if (rc == kTableCacheFull) break;                 // the rest goes into the next launch
            if (rc) return rc;
            last_ptr = ptr; last_nref = nr;
        }
        h_tab[j] = last_ptr;
        h_phase[j] = (float)(k0 * (double)dzs * ((double)n0 - (double)nr));
        h_fmax[j] = noprune ? p->Nx / 2 : live_fmax(p->Nx, (double)dx, k0 * (double)nr);
    }
    *i_done = i;
    if (i == i0) return BB_OK;
    int rc = ensure_steps(p, Nz);
    if (rc) return rc;
    const int ja = backward ? Nz - i : i0, n = i - i0;         // the steps touched are the range [ja, ja + n)
    BB_CUDA(cudaMemcpyAsync((void *)(p->d_htab + ja), h_tab.data() + ja, (size_t)n * sizeof(cf *), cudaMemcpyHostToDevice, s));
    BB_CUDA(cudaMemcpyAsync(p->d_phase + ja, h_phase.data() + ja, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s));
    BB_CUDA(cudaMemcpyAsync(p->d_fmax + ja, h_fmax.data() + ja, (size_t)n * sizeof(int), cudaMemcpyHostToDevice, s));
    return BB_OK;
}

int ws_reserve(Workspace &w, size_t bytes) {
    if (bytes <= w.bytes) return BB_OK;
    if (w.ptr) { cudaFree(w.ptr); w.ptr = nullptr; w.bytes = 0; }
    BB_CUDA(cudaMalloc(&w.ptr, bytes));
    w.bytes = bytes;
    return BB_OK;
}

int run_program(Plan *p, cf *field, int B, const bb::PhaseProg *prog, int nprog, cudaStream_t s) {
    KParams P;
    memset(&P, 0, sizeof P);
    P.field = field; P.Nx = p->Nx; P.Ny = p->Ny; P.B = B; P.BW = batch_warps(B);
    P.mode = 1;
    for (int i = 0; i < nprog; ++i) P.prog[i] = prog[i];
    P.twx = p->twx; P.twy = p->twy; P.bar = p->bar; P.status = p->status;
    P.p0 = 0; P.p1 = nprog;
    BB_CUDA(cudaMemsetAsync(p->bar, 0, sizeof(unsigned), s));
    cudaError_t e;
    if (p->k32) {
        e = bb::kernel_launch(p->Nx, p->Ny, P, p->grid, true, s);
    } else {
        // 2048-point lines: the 8-point-thread kernel, rows kept in natural kx order
        P.tw256 = p->tw256; P.twcx = p->twcx; P.twcy = p->twcy;
        P.xnat = 1;
        P.cw4 = p->Ny > 1024 ? 1 : 0;
        P.use_tma = !p->env_notma && make_field_tmap(&P.tmap, field, p->Nx, p->Ny, B, P.cw4 ? 4 : 8) ? 1 : 0;
        e = bb::kernel8_launch(p->Nx, p->Ny, P, p->grid, true, s);
    }
    ++g_launches;
    if (e != cudaSuccess) return fail(BB_ERR_CUDA, "cooperative launch failed: %s", cudaGetErrorString(e));
    return BB_OK;
}

}  // namespace

namespace bb {
#define BB_SWITCH_TX(fn, ...)                         \
    switch (Nx / 32) {                                \
        case 1: return inst1_##fn(__VA_ARGS__);       \
        case 2: return inst2_##fn(__VA_ARGS__);       \
        case 4: return inst4_##fn(__VA_ARGS__);       \
        case 8: return inst8_##fn(__VA_ARGS__);       \
        case 16: return inst16_##fn(__VA_ARGS__);     \
        case 32: return inst32_##fn(__VA_ARGS__);     \
    }
int kernel_prepare(int Nx, int Ny) {
    BB_SWITCH_TX(prepare, Ny / 32)
    return (int)cudaErrorInvalidValue;
}
int kernel_blocks_per_sm(int Nx, int Ny) {
    BB_SWITCH_TX(blocks_per_sm, Ny / 32)
    return 0;
}
cudaError_t kernel_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s) {
    BB_SWITCH_TX(launch, Ny / 32, P, grid, coop, s)
    return cudaErrorInvalidValue;
}
#define BB_SWITCH_PX(cw, bt, fn, ...)                                 \
    switch (Nx / 256) {                                               \
        case 1: return inst16_1_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 2: return inst16_2_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 4: return inst16_4_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 8: return inst16_8_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
    }
bool kernel16_supports(int Nx, int Ny) {
    auto ok = [](int n) { return n == 256 || n == 512 || n == 1024 || n == 2048; };
    return ok(Nx) && ok(Ny);
}
int kernel16_prepare(int Nx, int Ny) {
    auto f0 = [&]() -> cudaError_t { BB_SWITCH_PX(8, 0, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f1 = [&]() -> cudaError_t { BB_SWITCH_PX(4, 0, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f2 = [&]() -> cudaError_t { BB_SWITCH_PX(8, 1, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f3 = [&]() -> cudaError_t { BB_SWITCH_PX(4, 1, prepare, Ny / 256) return cudaErrorInvalidValue; };
    cudaError_t e = f0();
    if (e == cudaSuccess) e = f1();
    if (e == cudaSuccess) e = f2();
    if (e == cudaSuccess) e = f3();
    return (int)e;
}
int kernel16_blocks_per_sm(int Nx, int Ny) {
    auto f0 = [&]() -> int { BB_SWITCH_PX(8, 0, blocks_per_sm, Ny / 256) return 0; };
    auto f1 = [&]() -> int { BB_SWITCH_PX(4, 0, blocks_per_sm, Ny / 256) return 0; };
    auto f2 = [&]() -> int { BB_SWITCH_PX(8, 1, blocks_per_sm, Ny / 256) return 0; };
    auto f3 = [&]() -> int { BB_SWITCH_PX(4, 1, blocks_per_sm, Ny / 256) return 0; };
    return std::min(std::min(f0(), f1()), std::min(f2(), f3()));
}
cudaError_t kernel16_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s) {
    if (P.B > 1) {
        if (P.cw4) { BB_SWITCH_PX(4, 1, launch, Ny / 256, P, grid, coop, s) }
        else { BB_SWITCH_PX(8, 1, launch, Ny / 256, P, grid, coop, s) }
    } else {
        if (P.cw4) { BB_SWITCH_PX(4, 0, launch, Ny / 256, P, grid, coop, s) }
        else { BB_SWITCH_PX(8, 0, launch, Ny / 256, P, grid, coop, s) }
    }
    return cudaErrorInvalidValue;
}
#define BB_SWITCH_PX8(cw, bt, fn, ...)                               \
    switch (Nx / 256) {                                              \
        case 1: return inst8_1_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 2: return inst8_2_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 4: return inst8_4_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
        case 8: return inst8_8_cw##cw##_b##bt##_##fn(__VA_ARGS__);   \
    }
bool kernel8_supports(int Nx, int Ny) {
    auto ok = [](int n) { return n == 256 || n == 512 || n == 1024 || n == 2048; };
    return ok(Nx) && ok(Ny);
}
int kernel8_prepare(int Nx, int Ny) {
    auto f0 = [&]() -> cudaError_t { BB_SWITCH_PX8(8, 0, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f1 = [&]() -> cudaError_t { BB_SWITCH_PX8(4, 0, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f2 = [&]() -> cudaError_t { BB_SWITCH_PX8(8, 1, prepare, Ny / 256) return cudaErrorInvalidValue; };
    auto f3 = [&]() -> cudaError_t { BB_SWITCH_PX8(4, 1, prepare, Ny / 256) return cudaErrorInvalidValue; };
    cudaError_t e = f0();
    if (e == cudaSuccess) e = f1();
    if (e == cudaSuccess) e = f2();
    if (e == cudaSuccess) e = f3();
    return (int)e;
}
int kernel8_blocks_per_sm(int Nx, int Ny) {
    auto f0 = [&]() -> int { BB_SWITCH_PX8(8, 0, blocks_per_sm, Ny / 256) return 0; };
    auto f1 = [&]() -> int { BB_SWITCH_PX8(4, 0, blocks_per_sm, Ny / 256) return 0; };
    auto f2 = [&]() -> int { BB_SWITCH_PX8(8, 1, blocks_per_sm, Ny / 256) return 0; };
    auto f3 = [&]() -> int { BB_SWITCH_PX8(4, 1, blocks_per_sm, Ny / 256) return 0; };
    return std::min(std::min(f0(), f1()), std::min(f2(), f3()));
}
cudaError_t kernel8_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s) {
    if (P.B > 1) {
        if (P.cw4) { BB_SWITCH_PX8(4, 1, launch, Ny / 256, P, grid, coop, s) }
        else { BB_SWITCH_PX8(8, 1, launch, Ny / 256, P, grid, coop, s) }
    } else {
        if (P.cw4) { BB_SWITCH_PX8(4, 0, launch, Ny / 256, P, grid, coop, s) }
        else { BB_SWITCH_PX8(8, 0, launch, Ny / 256, P, grid, coop, s) }
    }
    return cudaErrorInvalidValue;
}
}  // namespace bb

// ==========================================================================================
extern "C" {

const char *bb_last_error(void) { return g_err.c_str(); }
const char *bb_last_kernel(void) { return g_last_kernel; }
int bb_version(void) { return 100; }
unsigned long long bb_launch_count(void) { return g_launches; }

void bb_shutdown(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    cudaDeviceSynchronize();
    for (Plan *p : g_plans) destroy_plan(p);
    g_plans.clear();
    for (auto &kv : g_ctx) {
        DeviceCtx &c = kv.second;
        for (Workspace *w : {&c.field, &c.dn, &c.I, &c.misc}) {
            if (w->ptr) cudaFree(w->ptr);
            w->ptr = nullptr; w->bytes = 0;
        }
        for (cudaEvent_t e : c.events) cudaEventDestroy(e);
        c.events.clear();
        for (cudaStream_t *st : {&c.s_in, &c.s_run, &c.s_out}) {
            if (*st) cudaStreamDestroy(*st);
            *st = nullptr;
        }
    }
    g_ctx.clear();
}

int bb_device_status(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return fail(BB_ERR_CUDA, "cudaDeviceSynchronize: %s", cudaGetErrorString(e));
    for (Plan *p : g_plans) {
        int st = 0;
        BB_CUDA(cudaMemcpy(&st, p->status, sizeof st, cudaMemcpyDeviceToHost));
        if (st != 0) {
            cudaMemset(p->status, 0, sizeof st);
            return fail(BB_ERR_INTERNAL, "grid barrier watchdog tripped (Nx=%d, Ny=%d)", p->Nx, p->Ny);
        }
    }
    return BB_OK;
}

}  // extern "C"
namespace {
// bb_propagate_ex without the lock (the helpers that are propagations in disguise call it too)
int propagate_impl(void *field, const float *dn, int Nx, int Ny, int Nz, float dx, float dz, float lambda,
                   float n0, float *intensity_out, const bb_opts *opts, bool allow_zero_dz = false) {
    int B; unsigned flags;
    int rc = validate_common(field, dn, Nx, Ny, Nz, dx, allow_zero_dz && dz == 0.f ? 1.f : dz, lambda, n0, opts, &B, &flags);
    if (rc) return rc;
    Plan *p;
    rc = get_plan(Nx, Ny, &p);
    if (rc) return rc;
    cudaStream_t s = opts ? (cudaStream_t)opts->stream : (cudaStream_t)0;
    const float *nref = opts ? opts->nref : nullptr;
    // A batch the batch variant of the 16-point-thread kernel cannot take (the screen factors of a CTA's rows
    // must fit one buffer) runs field by field on its single-field variant -- faster than the 32-point-thread
    // kernel, and the only way on a grid with a 2048-point side; dn is then read once per field.
    if (B > 1 && p->k16 && !use_k16(p, B) && !use_k8(p, B) && !use_kc(p, B)) {
        const size_t npx1 = (size_t)Nx * Ny;
        for (int b = 0; b < B; ++b) {
            bb_opts o = *opts;
            o.batch = 1;
            o.flags = flags & ~BB_INTENSITY_PER_FIELD;
            float *I = intensity_out;
            if (intensity_out && (flags & BB_INTENSITY_PER_FIELD)) I = intensity_out + (size_t)b * Nz * npx1;
            else if (b > 0) o.flags |= BB_ACCUMULATE;          // summed over the batch
            rc = propagate_impl((cf *)field + (size_t)b * npx1, dn, Nx, Ny, Nz, dx, dz, lambda, n0, I, &o, allow_zero_dz);
            if (rc) return rc;
        }
        return BB_OK;
    }
    choose_tile_width(p, B, Nz, dx, lambda, n0, nref);
    std::vector<const cf *> h_tab(Nz);
    std::vector<float> h_phase(Nz);
    double k0 = kTwoPi / (double)lambda;
    const bool backward = (flags & BB_BACKWARD) != 0;
    float phase_b = (float)(k0 * (double)(backward ? -dz : dz));
    size_t npx = (size_t)Nx * Ny;
    int i0 = 0;                                               // position in the processing order
    while (i0 < Nz) {
        int i1;
        rc = prepare_steps(p, B, Nz, i0, dx, dz, lambda, n0, nref, flags, s, h_tab, h_phase, &i1);
        if (rc) return rc;
        if (i1 <= i0) return fail(BB_ERR_OOM, "propagator table cache too small for one step");
        const int j0 = backward ? Nz - i1 : i0, j1 = backward ? Nz - i0 : i1;   // the steps of this launch
        rc = launch_steps(p, (cf *)field, dn ? dn + (size_t)j0 * npx : nullptr,
                          intensity_out ? intensity_out + (size_t)j0 * npx : nullptr,
                          (long long)Nz * (long long)npx, B, Nz, j0, j1, phase_b, flags, s);
        if (rc) return rc;
        i0 = i1;
    }
    return BB_OK;
}
}  // namespace
extern "C" {

int bb_propagate_ex(void *field, const float *dn, int Nx, int Ny, int Nz, float dx, float dz, float lambda,
                    float n0, float *intensity_out, const bb_opts *opts) {
    std::lock_guard<std::mutex> lk(g_mu);
    return propagate_impl(field, dn, Nx, Ny, Nz, dx, dz, lambda, n0, intensity_out, opts);
}

int bb_refocus(void *field, int Nx, int Ny, int batch, float dx, float dz, float lambda, float n, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!std::isfinite(dz)) return fail(BB_ERR_INVALID_ARG, "dz must be finite");
    bb_opts o;
    o.struct_size = (int)sizeof(bb_opts);
    o.batch = batch;
    o.nref = nullptr;
    o.flags = BB_HOMOGENEOUS | (dz < 0.f ? BB_BACKWARD : 0u);      // conj(H(|dz|)) = H(-|dz|), evanescent modes cut either way
    o.stream = stream;
    return propagate_impl(field, nullptr, Nx, Ny, 1, dx, std::fabs(dz), lambda, n, nullptr, &o, true);
}

int bb_propagate(void *field, const float *dn, int Nx, int Ny, int Nz, float dx, float dz, float lambda,
                 float n0, float *intensity_out) {
    return bb_propagate_ex(field, dn, Nx, Ny, Nz, dx, dz, lambda, n0, intensity_out, nullptr);
}

int bb_extract_tiles(const void *src, int elem, int Nx, int Ny, int Nplanes, const float *emitter_positions, int M,
                     float dx, int T, void *tiles_out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!src || !emitter_positions || !tiles_out) return fail(BB_ERR_INVALID_ARG, "src, emitter_positions or tiles_out is NULL");
    if (elem != 1 && elem != 2) return fail(BB_ERR_INVALID_ARG, "elem = %d must be 1 (float) or 2 (float pairs)", elem);
    if (Nx < 1 || Ny < 1 || Nplanes < 1 || M < 1 || M > 65535 || Nplanes > 65535)
        return fail(BB_ERR_INVALID_ARG, "Nx, Ny, Nplanes, M must be >= 1 (Nplanes, M <= 65535)");
    if (T < 1 || T > Nx || T > Ny) return fail(BB_ERR_INVALID_ARG, "tile size T = %d must be in [1, min(Nx, Ny)]", T);
    if (!(dx > 0.f) || !std::isfinite(dx)) return fail(BB_ERR_INVALID_ARG, "dx must be positive and finite");
    int dev, sms;
    int rc = check_arch(&dev, &sms);
    if (rc) return rc;
    dim3 grid(Nplanes, M);
    if (elem == 1)
        bb::extract_tiles_kernel<1><<<grid, 256, 0, (cudaStream_t)stream>>>((const float *)src, Nx, Ny, Nplanes, emitter_positions, M, (double)dx, T, (float *)tiles_out);
    else
        bb::extract_tiles_kernel<2><<<grid, 256, 0, (cudaStream_t)stream>>>((const float *)src, Nx, Ny, Nplanes, emitter_positions, M, (double)dx, T, (float *)tiles_out);
    ++g_launches;
    BB_CUDA(cudaGetLastError());
    return BB_OK;
}

int bb_lightsheet(int Nx, int Ny, float dx, float lambda, float n0, float NA, float z_focus, void *field_out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!field_out) return fail(BB_ERR_INVALID_ARG, "field_out is NULL");
    if (!(NA > 0.f) || !(dx > 0.f) || !(lambda > 0.f) || !(n0 > 0.f) || !std::isfinite(NA) || !std::isfinite(z_focus))
        return fail(BB_ERR_INVALID_ARG, "NA, dx, lambda, n0 must be positive and finite, z_focus finite");
    if (!shape_ok(Nx, Ny))
        return fail(BB_ERR_UNSUPPORTED_SHAPE, "Nx = %d, Ny = %d: both must be powers of two in [32, 2048], and both >= 256 if one is 2048", Nx, Ny);
    int dev, sms;
    int rc = check_arch(&dev, &sms);
    if (rc) return rc;
    const double w0 = (double)lambda / (3.14159265358979323846 * (double)NA);
    bb::gaussian_sheet_kernel<<<dim3((Nx + 127) / 128, Ny), 128, 0, (cudaStream_t)stream>>>((cf *)field_out, Nx, Ny, (double)dx, w0);
    ++g_launches;
    BB_CUDA(cudaGetLastError());
    // back-propagation of the waist by z_focus in the medium n0 (also cuts the evanescent ky, as the definition does)
    bb_opts o;
    o.struct_size = (int)sizeof(bb_opts);
    o.batch = 1;
    o.nref = nullptr;
    o.flags = BB_HOMOGENEOUS | (z_focus > 0.f ? BB_BACKWARD : 0u);
    o.stream = stream;
    return propagate_impl(field_out, nullptr, Nx, Ny, 1, dx, std::fabs(z_focus), lambda, n0, nullptr, &o, true);
}

int bb_image_formation(const float *source, int Nx, int Ny, const float *emitter_positions, int M, float dx,
                       const float *psf_tiles, int T, float *image_out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!source || !emitter_positions || !psf_tiles || !image_out) return fail(BB_ERR_INVALID_ARG, "a pointer argument is NULL");
    if (Nx < 1 || Ny < 1 || M < 1 || M > 65535) return fail(BB_ERR_INVALID_ARG, "Nx, Ny, M must be >= 1 (M <= 65535)");
    if (T < 1 || T > Nx || T > Ny || T > 96) return fail(BB_ERR_INVALID_ARG, "tile size T = %d must be in [1, min(Nx, Ny, 96)]", T);
    if (!(dx > 0.f) || !std::isfinite(dx)) return fail(BB_ERR_INVALID_ARG, "dx must be positive and finite");
    int dev, sms;
    int rc = check_arch(&dev, &sms);
    if (rc) return rc;
    DeviceCtx &ctx = device_ctx();
    const size_t own_bytes = (((size_t)Nx * Ny * sizeof(int)) + 255) & ~(size_t)255;
    rc = ws_reserve(ctx.misc, own_bytes + (size_t)M * (Nx + Ny) * sizeof(double));
    if (rc) return rc;
    int *owner = (int *)ctx.misc.ptr;
    double *dx2 = (double *)((char *)ctx.misc.ptr + own_bytes), *dy2 = dx2 + (size_t)M * Nx;
    cudaStream_t s = (cudaStream_t)stream;
    bb::emitter_axis_dist2_kernel<<<dim3((Nx + 127) / 128, M), 128, 0, s>>>(Nx, emitter_positions, 0, M, (double)dx, dx2);
    bb::emitter_axis_dist2_kernel<<<dim3((Ny + 127) / 128, M), 128, 0, s>>>(Ny, emitter_positions, 1, M, (double)dx, dy2);
    bb::nearest_emitter_kernel<<<dim3((Nx + 127) / 128, (Ny + 7) / 8), 128, 0, s>>>(Nx, Ny, M, dx2, dy2, owner);
    g_launches += 3;
    const size_t halo = (size_t)(32 + T - 1) * (8 + T - 1) * 8, tile = (size_t)T * T * sizeof(float);
    const int K = (int)std::max<size_t>(0, std::min<size_t>(16, ((size_t)160 * 1024 - halo) / tile));   // staged tiles per CTA
    const size_t smem = halo + (size_t)K * tile;
    if (smem > 48 * 1024)
        BB_CUDA(cudaFuncSetAttribute(bb::image_formation_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    bb::image_formation_kernel<<<dim3((Nx + 31) / 32, (Ny + 7) / 8), 256, smem, s>>>(source, owner, Nx, Ny, psf_tiles, T, K, image_out);
    ++g_launches;
    BB_CUDA(cudaGetLastError());
    return BB_OK;
}

}  // extern "C"
namespace {
int propagate_host_impl(void *field_host, const float *dn_host, int Nx, int Ny, int Nz, float dx, float dz,
                        float lambda, float n0, float *inten_host, const bb_opts *opts);
}
extern "C" {
int bb_propagate_host(void *field_host, const float *dn_host, int Nx, int Ny, int Nz, float dx, float dz,
                      float lambda, float n0, float *inten_host, const bb_opts *opts) {
    std::lock_guard<std::mutex> lk(g_mu);
    return propagate_host_impl(field_host, dn_host, Nx, Ny, Nz, dx, dz, lambda, n0, inten_host, opts);
}
}  // extern "C"
namespace {
int propagate_host_impl(void *field_host, const float *dn_host, int Nx, int Ny, int Nz, float dx, float dz,
                        float lambda, float n0, float *inten_host, const bb_opts *opts) {
    int B; unsigned flags;
    int rc = validate_common(field_host, dn_host, Nx, Ny, Nz, dx, dz, lambda, n0, opts, &B, &flags);
    if (rc) return rc;
    Plan *p;
    rc = get_plan(Nx, Ny, &p);
    if (rc) return rc;
    DeviceCtx &ctx = device_ctx();
    const float *nref = opts ? opts->nref : nullptr;
    // A batch the batch kernels cannot take runs field by field on the single-field kernel, as in propagate_impl --
    // but inside the chunk loop below, one launch per field on the resident dn chunk, so that every dn chunk crosses
    // PCIe once per call and the three streams keep running (not once per field with the streams drained in between).
    const bool fbf = B > 1 && p->k16 && !use_k16(p, B) && !use_k8(p, B) && !use_kc(p, B);
    const int LB = fbf ? 1 : B;                              // fields per launch
    choose_tile_width(p, LB, Nz, dx, lambda, n0, nref);
    const size_t npx = (size_t)Nx * Ny;
    const bool per_field = (flags & BB_INTENSITY_PER_FIELD) != 0;
    const bool backward = (flags & BB_BACKWARD) != 0;
    const int IB = per_field ? B : 1;                        // intensity volumes
    // z-chunks of ~32 MiB of dn, three buffers in flight per direction
    const int NBUF = 3;
    int CZ = (int)std::max<size_t>(1, ((size_t)32 << 20) / (npx * sizeof(float)));
    CZ = std::min(CZ, Nz);
    rc = ws_reserve(ctx.field, (size_t)B * npx * sizeof(cf));
    if (!rc && dn_host) rc = ws_reserve(ctx.dn, (size_t)NBUF * CZ * npx * sizeof(float));
    if (!rc && inten_host) rc = ws_reserve(ctx.I, (size_t)NBUF * IB * CZ * npx * sizeof(float));
    if (rc) return rc;
    cf *d_field = (cf *)ctx.field.ptr;
    float *d_dn = dn_host ? (float *)ctx.dn.ptr : nullptr;
    float *d_I = inten_host ? (float *)ctx.I.ptr : nullptr;

    // streams and events live as long as the library (bb_shutdown releases them)
    for (cudaStream_t *st : {&ctx.s_in, &ctx.s_run, &ctx.s_out})
        if (!*st) BB_CUDA(cudaStreamCreateWithFlags(st, cudaStreamNonBlocking));
    cudaStream_t s_in = ctx.s_in, s_run = ctx.s_run, s_out = ctx.s_out;
    const int nchunks = (Nz + CZ - 1) / CZ;
    while ((int)ctx.events.size() < 3 * nchunks) {
        cudaEvent_t e;
        BB_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx.events.push_back(e);
    }
    cudaEvent_t *ev_in = ctx.events.data(), *ev_run = ev_in + nchunks, *ev_out = ev_run + nchunks;
    int result = BB_OK;
    auto drain = [&]() { cudaStreamSynchronize(s_in); cudaStreamSynchronize(s_run); cudaStreamSynchronize(s_out); };
#define BB_TRY(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { result = fail(BB_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); drain(); return result; } } while (0)

    BB_TRY(cudaMemcpyAsync(d_field, field_host, (size_t)B * npx * sizeof(cf), cudaMemcpyHostToDevice, s_run));
    std::vector<const cf *> h_tab(Nz);
    std::vector<float> h_phase(Nz);
    double k0 = kTwoPi / (double)lambda;
    float phase_b = (float)(k0 * (double)(backward ? -dz : dz));
    int prepared = 0;                                        // positions [0, prepared) of the processing order have tables in place
    for (int c = 0; c < nchunks; ++c) {                      // c counts in processing order: backward runs start at the far end
        const int zc = backward ? nchunks - 1 - c : c;
        const int j0 = zc * CZ, j1 = std::min(Nz, j0 + CZ), nz = j1 - j0;
        const int buf = c % NBUF;
        float *dn_b = d_dn ? d_dn + (size_t)buf * CZ * npx : nullptr;
        float *I_b = d_I ? d_I + (size_t)buf * IB * CZ * npx : nullptr;
        if (dn_b) {
            // dn chunk in: the buffer is free once the chunk that last used it has been computed
            if (c >= NBUF) BB_TRY(cudaStreamWaitEvent(s_in, ev_run[c - NBUF], 0));
            BB_TRY(cudaMemcpyAsync(dn_b, dn_host + (size_t)j0 * npx, (size_t)nz * npx * sizeof(float),
                                   cudaMemcpyHostToDevice, s_in));
            BB_TRY(cudaEventRecord(ev_in[c], s_in));
            BB_TRY(cudaStreamWaitEvent(s_run, ev_in[c], 0));
        }
        if (I_b && c >= NBUF) BB_TRY(cudaStreamWaitEvent(s_run, ev_out[c - NBUF], 0));
        if (I_b && (flags & BB_ACCUMULATE)) {                // existing contents are part of the input
            for (int b = 0; b < IB; ++b)
                BB_TRY(cudaMemcpyAsync(I_b + (size_t)b * CZ * npx, inten_host + ((size_t)b * Nz + j0) * npx,
                                       (size_t)nz * npx * sizeof(float), cudaMemcpyHostToDevice, s_run));
        }
        const int ia = backward ? Nz - j1 : j0, ib = backward ? Nz - j0 : j1;      // positions of this chunk's steps
        int i = ia;
        while (i < ib) {
            if (i >= prepared) {
                rc = prepare_steps(p, LB, Nz, i, dx, dz, lambda, n0, nref, flags, s_run, h_tab, h_phase, &prepared);
                if (rc || prepared <= i) { drain(); return rc ? rc : fail(BB_ERR_OOM, "propagator table cache too small"); }
            }
            const int ie = std::min(ib, prepared);
            const int ja = backward ? Nz - ie : i, jb = backward ? Nz - i : ie;    // the steps of this launch
            for (int b = 0; b < (fbf ? B : 1); ++b) {
                float *I_l = I_b ? I_b + (size_t)(ja - j0) * npx : nullptr;
                unsigned fl = flags;
                if (fbf) {                                   // one field: its own volume, or added to the sum of the earlier ones
                    fl &= ~(unsigned)BB_INTENSITY_PER_FIELD;
                    if (per_field) { if (I_l) I_l += (size_t)b * CZ * npx; }
                    else if (b > 0) fl |= BB_ACCUMULATE;
                }
                rc = launch_steps(p, d_field + (fbf ? (size_t)b * npx : 0), dn_b ? dn_b + (size_t)(ja - j0) * npx : nullptr,
                                  I_l, (long long)CZ * (long long)npx, LB, Nz, ja, jb, phase_b, fl, s_run);
                if (rc) { drain(); return rc; }
            }
            i = ie;
        }
        BB_TRY(cudaEventRecord(ev_run[c], s_run));
        if (I_b) {
            BB_TRY(cudaStreamWaitEvent(s_out, ev_run[c], 0));
            for (int b = 0; b < IB; ++b)
                BB_TRY(cudaMemcpyAsync(inten_host + ((size_t)b * Nz + j0) * npx, I_b + (size_t)b * CZ * npx,
                                       (size_t)nz * npx * sizeof(float), cudaMemcpyDeviceToHost, s_out));
            BB_TRY(cudaEventRecord(ev_out[c], s_out));
        }
    }
    BB_TRY(cudaMemcpyAsync(field_host, d_field, (size_t)B * npx * sizeof(cf), cudaMemcpyDeviceToHost, s_run));
    BB_TRY(cudaStreamSynchronize(s_run));
    BB_TRY(cudaStreamSynchronize(s_out));
    BB_TRY(cudaStreamSynchronize(s_in));
    int st = 0;
    BB_TRY(cudaMemcpy(&st, p->status, sizeof st, cudaMemcpyDeviceToHost));
#undef BB_TRY
    if (st != 0) {
        cudaMemset(p->status, 0, sizeof st);
        return fail(BB_ERR_INTERNAL, "grid barrier watchdog tripped");
    }
    return result;
}

}  // namespace
extern "C" {

int bb_nref_from_dn(const float *dn, int Nx, int Ny, int Nz, float n0, int slab, float *nref_out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!dn || !nref_out) return fail(BB_ERR_INVALID_ARG, "dn_volume or nref_out is NULL");
    if (Nx < 1 || Ny < 1 || Nz < 1 || slab < 1) return fail(BB_ERR_INVALID_ARG, "Nx, Ny, Nz, slab must be >= 1");
    int dev, sms;
    int rc = check_arch(&dev, &sms);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const int NP = 16;
    DeviceCtx &ctx = device_ctx();
    rc = ws_reserve(ctx.misc, (size_t)Nz * NP * sizeof(double));
    if (rc) return rc;
    double *d_part = (double *)ctx.misc.ptr;
    size_t npx = (size_t)Nx * Ny;
    for (int j0 = 0; j0 < Nz; j0 += 32768) {                 // gridDim.y limit
        int nz = std::min(32768, Nz - j0);
        bb::slice_sum_kernel<<<dim3(NP, nz), 256, 0, s>>>(dn + (size_t)j0 * npx, npx, d_part + (size_t)j0 * NP);
        ++g_launches;
    }
    BB_CUDA(cudaGetLastError());
    std::vector<double> part((size_t)Nz * NP);
    BB_CUDA(cudaMemcpyAsync(part.data(), d_part, part.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
    BB_CUDA(cudaStreamSynchronize(s));
    for (int j0 = 0; j0 < Nz; j0 += slab) {
        int j1 = std::min(Nz, j0 + slab);
        long double sum = 0.0L;
        for (int j = j0; j < j1; ++j) {
            double sj = 0.0;
            for (int q = 0; q < NP; ++q) sj += part[(size_t)j * NP + q];
            sum += sj;
        }
        double mean = (double)(sum / ((long double)npx * (long double)(j1 - j0)));
        float v = (float)((double)n0 + mean);
        for (int j = j0; j < j1; ++j) nref_out[j] = v;
    }
    return BB_OK;
}

int bb_probe_trace(long long *device_buf, int phases) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_trace = device_buf;
    g_trace_phases = device_buf ? phases : 0;
    g_trace_dev = -1;
    if (device_buf) cudaGetDevice(&g_trace_dev);
    return BB_OK;
}

int bb_fft2(void *field, int Nx, int Ny, int batch, int sign, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!field) return fail(BB_ERR_INVALID_ARG, "field is NULL");
    if (batch < 1) return fail(BB_ERR_INVALID_ARG, "batch must be >= 1");
    if (sign != -1 && sign != 1) return fail(BB_ERR_INVALID_ARG, "sign must be -1 or +1");
    if (!shape_ok(Nx, Ny))
        return fail(BB_ERR_UNSUPPORTED_SHAPE, "Nx = %d, Ny = %d: both must be powers of two in [32, 2048], and both >= 256 if one is 2048", Nx, Ny);
    Plan *p;
    int rc = get_plan(Nx, Ny, &p);
    if (rc) return rc;
    bb::PhaseProg prog[2];
    if (sign < 0) {
        prog[0] = {1, 0, 1, 1.f};
        prog[1] = {0, 0, 1, 1.f};
    } else {
        prog[0] = {0, 1, 0, 1.f};
        prog[1] = {1, 1, 0, (float)(1.0 / ((double)Nx * (double)Ny))};
    }
    return run_program(p, (cf *)field, batch, prog, 2, (cudaStream_t)stream);
}

int bb_propagator_table(int Nx, int Ny, float dx, float dz, float lambda, float nref, void *out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!out) return fail(BB_ERR_INVALID_ARG, "table_out is NULL");
    if (!(dx > 0.f) || !(dz > 0.f) || !(lambda > 0.f) || !(nref > 0.f))
        return fail(BB_ERR_INVALID_ARG, "dx, dz, lambda, nref must be positive");
    if (!shape_ok(Nx, Ny))
        return fail(BB_ERR_UNSUPPORTED_SHAPE, "Nx = %d, Ny = %d: both must be powers of two in [32, 2048], and both >= 256 if one is 2048", Nx, Ny);
    Plan *p;
    int rc = get_plan(Nx, Ny, &p);
    if (rc) return rc;
    TableKey k = {dx, dz, lambda, nref, 1};
    return build_table(p, k, (cf *)out, (cudaStream_t)stream);
}

int bb_multiplex_psf(const float *pos, const float *phase, const float *amp, int M, float NA, int Nx, int Ny,
                     float dx, float lambda, void *field_out, void *stream) {
    return bb_multiplex_annular(pos, phase, amp, M, 0.f, NA, Nx, Ny, dx, lambda, field_out, stream);
}

int bb_multiplex_annular(const float *pos, const float *phase, const float *amp, int M, float NA_in, float NA, int Nx, int Ny,
                         float dx, float lambda, void *field_out, void *stream) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!pos || !field_out) return fail(BB_ERR_INVALID_ARG, "emitter_positions or field_out is NULL");
    if (M < 1) return fail(BB_ERR_INVALID_ARG, "M = %d must be >= 1", M);
    if (!(NA > 0.f) || !(dx > 0.f) || !(lambda > 0.f) || !std::isfinite(NA))
        return fail(BB_ERR_INVALID_ARG, "NA, dx, lambda must be positive and finite");
    if (!(NA_in >= 0.f) || !(NA_in <= NA)) return fail(BB_ERR_INVALID_ARG, "NA_inner must be in [0, NA]");
    if (!shape_ok(Nx, Ny))
        return fail(BB_ERR_UNSUPPORTED_SHAPE, "Nx = %d, Ny = %d: both must be powers of two in [32, 2048], and both >= 256 if one is 2048", Nx, Ny);
    Plan *p;
    int rc = get_plan(Nx, Ny, &p);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    // pupil pixel count, in double, same expression as the kernel's inside test
    const double ddx = dx, k0 = kTwoPi / (double)lambda, kc2 = (k0 * (double)NA) * (k0 * (double)NA);
    const double ki2 = (k0 * (double)NA_in) * (k0 * (double)NA_in);
    if (!(p->pupil.dx == dx && p->pupil.lambda == lambda && p->pupil.na_in == NA_in && p->pupil.na == NA)) {
        long long count = 0;
        std::vector<double> kx2(Nx), ky2(Ny);
        for (int i = 0; i < Nx; ++i) { int f = (i < Nx / 2) ? i : i - Nx; double k = kTwoPi * (double)f / ((double)Nx * ddx); kx2[i] = k * k; }
        for (int i = 0; i < Ny; ++i) { int f = (i < Ny / 2) ? i : i - Ny; double k = kTwoPi * (double)f / ((double)Ny * ddx); ky2[i] = k * k; }
        for (int q = 0; q < Ny; ++q)
            for (int i = 0; i < Nx; ++i)
                if (kx2[i] + ky2[q] <= kc2 && kx2[i] + ky2[q] >= ki2) ++count;
        // bounding box of the pupil in DFT bins: [-F, F] per axis, clipped to [-N/2, N/2 - 1]
        auto extent = [&](const std::vector<double> &k2, int N, int *lo, int *w) {
            int F = 0;
            for (int f = 0; f <= N / 2; ++f)
                if (k2[f] <= kc2) F = f;
            *lo = std::min(F, N / 2);
            *w = *lo + std::min(F, N / 2 - 1) + 1;
        };
        Plan::Pupil pu;
        pu.dx = dx; pu.lambda = lambda; pu.na_in = NA_in; pu.na = NA; pu.count = count;
        extent(kx2, Nx, &pu.Fx, &pu.Wx);
        extent(ky2, Ny, &pu.Fy, &pu.Wy);
        p->pupil = pu;
    }
    const long long count = p->pupil.count;
    if (count == 0) return fail(BB_ERR_INVALID_ARG, "pupil of NA = %g contains no grid frequency", (double)NA);
    const int Fx = p->pupil.Fx, Wx = p->pupil.Wx, Fy = p->pupil.Fy, Wy = p->pupil.Wy;
    const size_t em_bytes = (((size_t)M * sizeof(bb::EmitterPrep)) + 255) & ~(size_t)255;
    DeviceCtx &ctx = device_ctx();
    rc = ws_reserve(ctx.misc, em_bytes + (size_t)M * (Wx + Wy) * sizeof(cf) + 4096);
    if (rc) return rc;
    bb::EmitterPrep *em = (bb::EmitterPrep *)ctx.misc.ptr;
    cf *EX = (cf *)((char *)ctx.misc.ptr + em_bytes), *EY = EX + (size_t)M * Wx;
    bb::emitter_prep_kernel<<<(M + 127) / 128, 128, 0, s>>>(pos, phase, amp, M, Nx, Ny, ddx, em);
    ++g_launches;
    bb::emitter_axis_kernel<<<dim3((std::max(Wx, Wy) + 127) / 128, M), 128, 0, s>>>(em, M, Fx, Wx, Fy, Wy, EX, EY);
    ++g_launches;
    BB_CUDA(cudaMemsetAsync(field_out, 0, (size_t)Nx * Ny * sizeof(cf), s));
    bb::multiplex_gemm_kernel<<<dim3((Wx + 31) / 32, (Wy + 31) / 32), 256, 0, s>>>((cf *)field_out, Nx, Ny, ddx, ki2, kc2, EX, EY,
                                                                                   M, Fx, Wx, Fy, Wy);
    ++g_launches;
    BB_CUDA(cudaGetLastError());
    bb::PhaseProg prog[2];
    prog[0] = {0, 1, 0, 1.f};
    prog[1] = {1, 1, 0, (float)(1.0 / (double)count)};
    return run_program(p, (cf *)field_out, 1, prog, 2, s);
}

}  // extern "C"

// Hooks for the library's other translation units (bb_hooks.h).
#include "bb_hooks.h"
namespace bb {
int report_error(int code, const char *message) { return fail(code, "%s", message); }
void count_launches(unsigned n) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_launches += n;
}
}  // namespace bb
