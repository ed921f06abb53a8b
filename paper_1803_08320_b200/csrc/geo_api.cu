// geo_api.cu -- the C ABI of include/geo.h: argument validation, launch configuration, host-buffer
// convenience path.  No arithmetic of the method lives here; it is all in geo_kernel.cuh / geo_rhs.cuh.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/geo.h"
#include "../../include/geo_dev.h"
#include "geo_kernel.cuh"
#include "geo_rk45.cuh"
#include "geo_tab.cuh"
#include "geo_tabg.cuh"
#include "geo_ks.cuh"
#include "geo_ks_rk45.cuh"

using namespace geo;

struct geo_ctx {
    int metric;
    double M, a;
    int device;
    int sm_count;
    unsigned long long* counter;   // device: work-queue heads [2] (one per host-path slot; geo_integrate uses [0])
    // device scratch of geo_integrate_host (grow-only)
    void* scratch;
    size_t scratch_bytes;
    cudaStream_t host_stream[2];
    // GEO_TABULATED: the table in the kernel's node-major layout (device, owned)
    double4* tabA;
    double* tabB;
    TabMetric tm;
    // GEO_TABULATED_GENERAL: ten-field node records (device, owned)
    double* tabG;
    TabgMetric tgm;
    char err[256];
};

namespace {

typedef void (*kernel_fn)(const Params);

template <bool KERR, int SNAP>
kernel_fn pick_plain(bool plain) {
    return plain ? (kernel_fn)geo_rk4_kernel<KERR, SNAP, true, false> : (kernel_fn)geo_rk4_kernel<KERR, SNAP, false, false>;
}
template <bool KERR>
kernel_fn pick_snap(int snap, bool plain, bool wide, bool big) {
    if (big) {
        if (snap == SNAP_NONE) return plain ? (kernel_fn)geo_rk4_kernel<KERR, SNAP_NONE, true, false, true> : (kernel_fn)geo_rk4_kernel<KERR, SNAP_NONE, false, false, true>;
        return plain ? (kernel_fn)geo_rk4_kernel<KERR, SNAP_DIRECT, true, false, true> : (kernel_fn)geo_rk4_kernel<KERR, SNAP_DIRECT, false, false, true>;
    }
    switch (snap) {
        case SNAP_NONE:
            if (wide) return plain ? (kernel_fn)geo_rk4_kernel<KERR, SNAP_NONE, true, true> : (kernel_fn)geo_rk4_kernel<KERR, SNAP_NONE, false, true>;
            return pick_plain<KERR, SNAP_NONE>(plain);
        case SNAP_DIRECT: return pick_plain<KERR, SNAP_DIRECT>(plain);
        default: return pick_plain<KERR, SNAP_STAGED>(plain);
    }
}
kernel_fn pick_kernel(int metric, int snap, bool plain, bool wide, bool big) {
    return metric == GEO_KERR ? pick_snap<true>(snap, plain, wide, big) : pick_snap<false>(snap, plain, wide, big);
}

int fail(geo_ctx* ctx, int code, const char* msg) {
    if (ctx) snprintf(ctx->err, sizeof ctx->err, "%s", msg);
    return code;
}
int fail_cuda(geo_ctx* ctx, cudaError_t e, const char* what) {
    if (ctx) snprintf(ctx->err, sizeof ctx->err, "%s: %s", what, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? GEO_ENOMEM : GEO_ECUDA;
}

// A ctx belongs to the device that was current at geo_create: its counters, scratch, tables and SM count are that
// device's.  Every entry point runs with that device current and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
        else if (err == cudaSuccess) prev = -1;      // nothing to restore
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};
#define GEO_ON_CTX_DEVICE(ctx)                                                         \
    DeviceGuard device_guard_((ctx)->device);                                          \
    if (device_guard_.err != cudaSuccess) return fail_cuda((ctx), device_guard_.err, "cudaSetDevice(ctx device)")

bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

int popcount8(uint32_t m) {
    int c = 0;
    for (int k = 0; k < 8; ++k) c += (m >> k) & 1u;
    return c;
}

// Argument checks shared by the device and host entry points.  Returns GEO_OK or GEO_EINVAL.
int validate(geo_ctx* ctx, const double* state_in, int64_t n, double h, int64_t nsteps, const geo_stop* stop,
             int64_t snapshot_every, const geo_out* out, bool check_align) {
    if (!ctx) return GEO_EINVAL;
    ctx->err[0] = 0;
    if (!stop || !out) return fail(ctx, GEO_EINVAL, "stop and out must not be NULL");
    if (n < 0 || nsteps < 0 || snapshot_every < 0) return fail(ctx, GEO_EINVAL, "n, nsteps, snapshot_every must be >= 0");
    if (nsteps > 0x7fffffffLL) return fail(ctx, GEO_EINVAL, "nsteps must be < 2^31");
    if (!std::isfinite(h) || h == 0.0) return fail(ctx, GEO_EINVAL, "h must be finite and non-zero");
    if (stop->kind != GEO_TIMELIKE && stop->kind != GEO_NULL) return fail(ctx, GEO_EINVAL, "stop.kind must be GEO_TIMELIKE or GEO_NULL");
    if (std::isnan(stop->r_capture) || std::isnan(stop->r_escape)) return fail(ctx, GEO_EINVAL, "stop radii must not be NaN");
    if (stop->flags & ~(GEO_FLAG_PLAIN_UPDATE | GEO_FLAG_STATIC_MAP | GEO_FLAG_STAGED_SNAP | GEO_FLAG_CARTESIAN_SNAP | GEO_FLAG_TAB_GATHER)) return fail(ctx, GEO_EINVAL, "unknown stop.flags bit");
    if (ctx->metric == GEO_TABULATED || ctx->metric == GEO_TABULATED_GENERAL) {
        const int32_t ok = GEO_FLAG_PLAIN_UPDATE | GEO_FLAG_TAB_GATHER;
        if (stop->flags & ~ok) return fail(ctx, GEO_EINVAL, "tabulated metrics: only GEO_FLAG_PLAIN_UPDATE and GEO_FLAG_TAB_GATHER are supported");
    }
    if (ctx->metric == GEO_KERR_SCHILD) {
        const int32_t ok = GEO_FLAG_PLAIN_UPDATE | GEO_FLAG_STATIC_MAP;
        if (stop->flags & ~ok) return fail(ctx, GEO_EINVAL, "GEO_KERR_SCHILD: only GEO_FLAG_PLAIN_UPDATE and GEO_FLAG_STATIC_MAP are supported (records are Cartesian already)");
    }
    if (n == 0) return GEO_OK;
    if (!state_in || !out->final_state || !out->status || !out->steps_done) return fail(ctx, GEO_EINVAL, "state_in, final_state, status, steps_done are required");
    if (snapshot_every > 0) {
        if (!out->snapshots || !out->snap_count) return fail(ctx, GEO_EINVAL, "snapshot_every > 0 needs snapshots and snap_count");
        if (out->snap_capacity < 1) return fail(ctx, GEO_EINVAL, "snap_capacity must be >= 1");
        if ((out->snap_mask & 0xFFu) == 0 || (out->snap_mask & ~0xFFu)) return fail(ctx, GEO_EINVAL, "snap_mask must select 1..8 of the 8 components");
    }
    if (check_align) {
        if (misaligned(state_in) || misaligned(out->final_state) || misaligned(out->status) || misaligned(out->steps_done) ||
            misaligned(out->eq_cross_r) || misaligned(out->health) || misaligned(out->snapshots) || misaligned(out->snap_count))
            return fail(ctx, GEO_EINVAL, "device pointers must be 16-byte aligned");
    }
    return GEO_OK;
}

struct LaunchPlan {
    kernel_fn fn;
    int snap_mode;
    int use_queue;
    int grid;
    int block;
    size_t smem;
    int ctas_per_sm;
    int regs;
};

int plan_launch(geo_ctx* ctx, int64_t n, int32_t flags, int64_t snapshot_every, int ncomp, LaunchPlan* lp) {
    // The direct writer (256-bit stores from registers) is the default at every cadence: since round 2 the record logic
    // sits behind the stepping loop's single rare-event branch and no longer costs the accepted step any registers
    // (round 1 routed snapshot_every >= 16 through the staged writer because the inlined record code made the Kerr
    // stepping loop spill: config 2 ran 319 ms direct / 188 ms staged; now 173 / 176 ms).
    const bool staged = (flags & GEO_FLAG_STAGED_SNAP) != 0;
    lp->snap_mode = snapshot_every > 0 ? (staged ? SNAP_STAGED : SNAP_DIRECT) : SNAP_NONE;
    // a batch without records that fits on the machine at 2 CTAs per SM runs the high-ILP instantiation (geo_kernel.cuh: WIDE)
    const bool wide = lp->snap_mode == SNAP_NONE && n <= (int64_t)ctx->sm_count * 2 * kBlock;
    // a batch that fits in ONE wave (n <= 512 x SMs) runs ONE CTA per SM of 128 k threads, k = ceil(n / (128 SMs)) = the
    // warps per scheduler it needs anyway (geo_kernel.cuh: BIG; the WIDE instantiation takes up to 256 threads): warps of
    // one CTA have the same age and progress evenly, several CTAs per SM do not (measured: DESIGN.md section 9)
    const int64_t k64 = (n + (int64_t)ctx->sm_count * kBlock - 1) / ((int64_t)ctx->sm_count * kBlock);
    const int k = k64 < 1 ? 1 : (k64 > 1024 ? 1024 : (int)k64);
    const bool one_wave = k <= kBigBlock / kBlock && lp->snap_mode != SNAP_STAGED;
    const bool big = one_wave && !wide && k >= 2;
    const int blk = one_wave ? k * kBlock : kBlock;
    lp->block = blk;
    lp->fn = pick_kernel(ctx->metric, lp->snap_mode, (flags & GEO_FLAG_PLAIN_UPDATE) != 0, wide, big);
    lp->smem = lp->snap_mode == SNAP_STAGED ? (size_t)kBlock * stage_stride(ncomp) * sizeof(double) : 0;
    lp->use_queue = (flags & GEO_FLAG_STATIC_MAP) ? 0 : 1;
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, (const void*)lp->fn);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncGetAttributes");
    lp->regs = fa.numRegs;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)lp->fn, lp->block, lp->smem);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    lp->ctas_per_sm = per_sm;
    const int64_t need = (n + lp->block - 1) / lp->block;
    if (lp->use_queue) {
        // persistent grid: every SM full, no more CTAs than there is work
        const int64_t resident = (int64_t)ctx->sm_count * per_sm;
        lp->grid = (int)(need < resident ? need : resident);
    } else {
        if (need > 0x7fffffffLL) return fail(ctx, GEO_EINVAL, "n too large for the static mapping");
        lp->grid = (int)need;
    }
    return GEO_OK;
}

typedef void (*tab_kernel_fn)(const TabParams);
tab_kernel_fn pick_tab_kernel(int32_t flags, bool snap = false) {
    const bool plain = (flags & GEO_FLAG_PLAIN_UPDATE) != 0;
    if (flags & GEO_FLAG_TAB_GATHER)
        return snap ? (plain ? (tab_kernel_fn)geo_tab_rk4_kernel<true, false, true> : (tab_kernel_fn)geo_tab_rk4_kernel<false, false, true>)
                    : (plain ? (tab_kernel_fn)geo_tab_rk4_kernel<true, false, false> : (tab_kernel_fn)geo_tab_rk4_kernel<false, false, false>);
    return snap ? (plain ? (tab_kernel_fn)geo_tab_rk4_kernel<true, true, true> : (tab_kernel_fn)geo_tab_rk4_kernel<false, true, true>)
                : (plain ? (tab_kernel_fn)geo_tab_rk4_kernel<true, true, false> : (tab_kernel_fn)geo_tab_rk4_kernel<false, true, false>);
}
size_t tab_smem(int32_t flags) { return (flags & GEO_FLAG_TAB_GATHER) ? 0 : (size_t)kTabSmemRows * kTabBlock * sizeof(double); }

int plan_tab(geo_ctx* ctx, int64_t n, int32_t flags, int* grid, int* per_sm_out, int* regs, bool snap = false) {
    tab_kernel_fn fn = pick_tab_kernel(flags, snap);
    int per_sm = 0;
    cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tab_smem(flags));
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncSetAttribute(smem)");
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, kTabBlock, tab_smem(flags));
    if (e != cudaSuccess) return fail_cuda(ctx, e, "occupancy(tab)");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, (const void*)fn);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncGetAttributes");
    const int64_t need = (n + kTabBlock - 1) / kTabBlock, resident = (int64_t)ctx->sm_count * per_sm;
    *grid = (int)(need < resident ? need : resident);
    *per_sm_out = per_sm;
    *regs = fa.numRegs;
    return GEO_OK;
}

int launch_tab(geo_ctx* ctx, const double* d_in, int64_t n, double h, int64_t nsteps, const geo_stop* stop,
               int64_t snapshot_every, const geo_out* out, cudaStream_t stream, unsigned long long* counter) {
    int grid = 0, per_sm = 0, regs = 0;
    const bool snap = snapshot_every > 0;
    int rc = plan_tab(ctx, n, stop->flags, &grid, &per_sm, &regs, snap);
    if (rc != GEO_OK) return rc;
    TabParams p;
    memset(&p, 0, sizeof p);
    p.in = d_in;
    p.n = n;
    p.h = h;
    p.h_half = h / 2.0;
    p.h_sixth = h / 6.0;
    p.nsteps = (int)nsteps;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.counter = counter;
    p.snap_every = (int)(snapshot_every > 0x7fffffffLL ? 0x7fffffffLL : snapshot_every);
    p.snap_cap = snap ? out->snap_capacity : 0;
    p.snap_mask = snap ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = snap ? popcount8(out->snap_mask) : 0;
    p.snaps = snap ? out->snapshots : nullptr;
    p.snap_count = snap ? out->snap_count : nullptr;
    p.m = ctx->tm;
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    pick_tab_kernel(stop->flags, snap)<<<grid, kTabBlock, tab_smem(stop->flags), stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

typedef void (*tabg_kernel_fn)(const TabgParams);
tabg_kernel_fn pick_tabg_kernel(int32_t flags, bool snap = false) {
    const bool plain = (flags & GEO_FLAG_PLAIN_UPDATE) != 0;
    if (flags & GEO_FLAG_TAB_GATHER)
        return snap ? (plain ? (tabg_kernel_fn)geo_tabg_rk4_kernel<true, false, true> : (tabg_kernel_fn)geo_tabg_rk4_kernel<false, false, true>)
                    : (plain ? (tabg_kernel_fn)geo_tabg_rk4_kernel<true, false, false> : (tabg_kernel_fn)geo_tabg_rk4_kernel<false, false, false>);
    return snap ? (plain ? (tabg_kernel_fn)geo_tabg_rk4_kernel<true, true, true> : (tabg_kernel_fn)geo_tabg_rk4_kernel<false, true, true>)
                : (plain ? (tabg_kernel_fn)geo_tabg_rk4_kernel<true, true, false> : (tabg_kernel_fn)geo_tabg_rk4_kernel<false, true, false>);
}
int tabg_block(int32_t flags) { return (flags & GEO_FLAG_TAB_GATHER) ? kTabBlock : kTabgCacheBlock; }
size_t tabg_smem(int32_t flags) { return (flags & GEO_FLAG_TAB_GATHER) ? 0 : (size_t)kTabgCacheRows * kTabgCacheBlock * sizeof(double); }

int plan_tabg(geo_ctx* ctx, int64_t n, int32_t flags, int* grid, int* per_sm_out, int* regs, bool snap = false) {
    tabg_kernel_fn fn = pick_tabg_kernel(flags, snap);
    int per_sm = 0;
    const int block = tabg_block(flags);
    cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tabg_smem(flags));
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncSetAttribute(smem)");
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, block, tabg_smem(flags));
    if (e != cudaSuccess) return fail_cuda(ctx, e, "occupancy(tabg)");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, (const void*)fn);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncGetAttributes");
    const int64_t need = (n + block - 1) / block, resident = (int64_t)ctx->sm_count * per_sm;
    *grid = (int)(need < resident ? need : resident);
    *per_sm_out = per_sm;
    *regs = fa.numRegs;
    return GEO_OK;
}

int launch_tabg(geo_ctx* ctx, const double* d_in, int64_t n, double h, int64_t nsteps, const geo_stop* stop,
                int64_t snapshot_every, const geo_out* out, cudaStream_t stream, unsigned long long* counter) {
    int grid = 0, per_sm = 0, regs = 0;
    const bool snap = snapshot_every > 0;
    int rc = plan_tabg(ctx, n, stop->flags, &grid, &per_sm, &regs, snap);
    if (rc != GEO_OK) return rc;
    TabgParams p;
    memset(&p, 0, sizeof p);
    p.in = d_in;
    p.n = n;
    p.h = h;
    p.h_half = h / 2.0;
    p.h_sixth = h / 6.0;
    p.nsteps = (int)nsteps;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.counter = counter;
    p.snap_every = (int)(snapshot_every > 0x7fffffffLL ? 0x7fffffffLL : snapshot_every);
    p.snap_cap = snap ? out->snap_capacity : 0;
    p.snap_mask = snap ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = snap ? popcount8(out->snap_mask) : 0;
    p.snaps = snap ? out->snapshots : nullptr;
    p.snap_count = snap ? out->snap_count : nullptr;
    p.m = ctx->tgm;
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    pick_tabg_kernel(stop->flags, snap)<<<grid, tabg_block(stop->flags), tabg_smem(stop->flags), stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

typedef void (*ks_kernel_fn)(const KsParams);
ks_kernel_fn pick_ks_kernel(bool snap, bool plain) {
    if (snap) return plain ? (ks_kernel_fn)geo_ks_rk4_kernel<SNAP_DIRECT, true> : (ks_kernel_fn)geo_ks_rk4_kernel<SNAP_DIRECT, false>;
    return plain ? (ks_kernel_fn)geo_ks_rk4_kernel<SNAP_NONE, true> : (ks_kernel_fn)geo_ks_rk4_kernel<SNAP_NONE, false>;
}

int plan_ks(geo_ctx* ctx, int64_t n, int32_t flags, bool snap, ks_kernel_fn* fn_out, int* grid, int* per_sm_out, int* regs) {
    ks_kernel_fn fn = pick_ks_kernel(snap, (flags & GEO_FLAG_PLAIN_UPDATE) != 0);
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, (const void*)fn);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaFuncGetAttributes");
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, kBlock, 0);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    const int64_t need = (n + kBlock - 1) / kBlock;
    if (flags & GEO_FLAG_STATIC_MAP) {
        if (need > 0x7fffffffLL) return fail(ctx, GEO_EINVAL, "n too large for the static mapping");
        *grid = (int)need;
    } else {
        const int64_t resident = (int64_t)ctx->sm_count * per_sm;
        *grid = (int)(need < resident ? need : resident);
    }
    if (fn_out) *fn_out = fn;
    if (per_sm_out) *per_sm_out = per_sm;
    if (regs) *regs = fa.numRegs;
    return GEO_OK;
}

// GEO_KERR_SCHILD: Kerr in Cartesian Kerr-Schild coordinates (geo_ks.cuh).
int launch_ks(geo_ctx* ctx, const double* d_in, int64_t n, double h, int64_t nsteps, const geo_stop* stop,
              int64_t snapshot_every, const geo_out* out, cudaStream_t stream, unsigned long long* counter) {
    ks_kernel_fn fn;
    int grid = 0;
    int rc = plan_ks(ctx, n, stop->flags, snapshot_every > 0, &fn, &grid, nullptr, nullptr);
    if (rc != GEO_OK) return rc;
    KsParams p;
    memset(&p, 0, sizeof p);
    p.in = d_in;
    p.n = n;
    p.h = h;
    p.h_half = h / 2.0;
    p.h_sixth = h / 6.0;
    p.nsteps = (int)nsteps;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    const double a2 = ctx->a * ctx->a;
    // end-point triggers (geo_ks.cuh): r^2 <= R^2 <= r^2 + a^2.  r_capture <= 0 never captures a finite point, +inf always
    // does (decided at y0); r_escape = +inf never escapes, r_escape <= 0 always triggers (decided behind the branch)
    p.cap_R2 = stop->r_capture > 0.0 ? stop->r_capture * stop->r_capture + a2 : -INFINITY;
    p.esc_R2 = stop->r_escape > 0.0 ? stop->r_escape * stop->r_escape : -1.0;
    p.use_queue = (stop->flags & GEO_FLAG_STATIC_MAP) ? 0 : 1;
    p.snap_every = (int)(snapshot_every > 0x7fffffffLL ? 0x7fffffffLL : snapshot_every);
    p.snap_cap = snapshot_every > 0 ? out->snap_capacity : 0;
    p.snap_mask = snapshot_every > 0 ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = snapshot_every > 0 ? popcount8(out->snap_mask) : 0;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.snaps = out->snapshots;
    p.snap_count = out->snap_count;
    p.counter = counter;
    p.bh.M = ctx->M;
    p.bh.a = ctx->a;
    p.bh.a2 = a2;
    p.bh.twoM = 2.0 * ctx->M;
    p.bh.four_a2 = 4.0 * a2;
    cudaError_t e;
    if (p.use_queue) {
        e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    }
    fn<<<grid, kBlock, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

int launch(geo_ctx* ctx, const double* d_in, int64_t n, double h, int64_t nsteps, const geo_stop* stop,
           int64_t snapshot_every, const geo_out* out, cudaStream_t stream, unsigned long long* counter) {
    if (ctx->metric == GEO_TABULATED) return launch_tab(ctx, d_in, n, h, nsteps, stop, snapshot_every, out, stream, counter);
    if (ctx->metric == GEO_TABULATED_GENERAL) return launch_tabg(ctx, d_in, n, h, nsteps, stop, snapshot_every, out, stream, counter);
    if (ctx->metric == GEO_KERR_SCHILD) return launch_ks(ctx, d_in, n, h, nsteps, stop, snapshot_every, out, stream, counter);
    const int ncomp = snapshot_every > 0 ? popcount8(out->snap_mask) : 0;
    LaunchPlan lp;
    int rc = plan_launch(ctx, n, stop->flags, snapshot_every, ncomp, &lp);
    if (rc != GEO_OK) return rc;

    Params p;
    memset(&p, 0, sizeof p);
    p.in = d_in;
    p.n = n;
    p.h = h;
    p.h_half = h / 2.0;
    p.h_sixth = h / 6.0;
    p.nsteps = (int)nsteps;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    p.use_queue = lp.use_queue;
    p.snap_every = (int)(snapshot_every > 0x7fffffffLL ? 0x7fffffffLL : snapshot_every);
    p.snap_cap = snapshot_every > 0 ? out->snap_capacity : 0;
    p.snap_mask = snapshot_every > 0 ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = ncomp;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.snaps = out->snapshots;
    p.snap_count = out->snap_count;
    p.coarse_steps = out->coarse_steps;
    p.counter = counter;
    p.bh.M = ctx->M;
    p.bh.a = ctx->a;
    p.bh.a2 = ctx->a * ctx->a;
    p.bh.twoM = 2.0 * ctx->M;
    p.bh.twoMa = 2.0 * ctx->M * ctx->a;
    fill_trig_consts(p.bh.tc);
    p.cartesian = (stop->flags & GEO_FLAG_CARTESIAN_SNAP) ? 1 : 0;

    cudaError_t e;
    if (lp.use_queue) {
        e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    }
    lp.fn<<<lp.grid, lp.block, lp.smem, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" {

int geo_create(geo_ctx** out_ctx, int metric, double M, double a) {
    if (!out_ctx) return GEO_EINVAL;
    *out_ctx = nullptr;
    if (metric != GEO_SCHWARZSCHILD && metric != GEO_KERR && metric != GEO_KERR_SCHILD) return GEO_EINVAL;
    if (!(M > 0.0) || !std::isfinite(M) || !(std::fabs(a) <= M)) return GEO_EINVAL;
    if (metric == GEO_SCHWARZSCHILD && a != 0.0) return GEO_EINVAL;
    geo_ctx* ctx = new (std::nothrow) geo_ctx;
    if (!ctx) return GEO_ENOMEM;
    memset(ctx, 0, sizeof *ctx);
    ctx->metric = metric;
    ctx->M = M;
    ctx->a = a;
    cudaError_t e = cudaGetDevice(&ctx->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->counter, 2 * sizeof(unsigned long long));
    if (e != cudaSuccess) {
        int rc = e == cudaErrorMemoryAllocation ? GEO_ENOMEM : GEO_ECUDA;
        delete ctx;
        return rc;
    }
    *out_ctx = ctx;
    return GEO_OK;
}

int geo_create_tabulated(geo_ctx** out_ctx, const geo_table* tb) {
    if (!out_ctx) return GEO_EINVAL;
    *out_ctx = nullptr;
    if (!tb || !tb->tab || tb->n1 < 4 || tb->n2 < 4 || tb->n1 > 0x3fffffff || tb->n2 > 0x3fffffff) return GEO_EINVAL;
    if (!(tb->d1 > 0.0) || !(tb->d2 > 0.0) || !std::isfinite(tb->d1) || !std::isfinite(tb->d2) ||
        !std::isfinite(tb->x1_0) || !std::isfinite(tb->x2_0))
        return GEO_EINVAL;
    geo_ctx* ctx = new (std::nothrow) geo_ctx;
    if (!ctx) return GEO_ENOMEM;
    memset(ctx, 0, sizeof *ctx);
    ctx->metric = GEO_TABULATED;
    ctx->M = NAN;
    ctx->a = NAN;
    const size_t nodes = (size_t)tb->n1 * (size_t)tb->n2;
    double* raw = nullptr;
    cudaError_t e = cudaGetDevice(&ctx->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->counter, 2 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->tabA, nodes * sizeof(double4));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->tabB, nodes * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&raw, 5 * nodes * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(raw, tb->tab, 5 * nodes * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        tab_pack_kernel<<<(unsigned)((nodes + 255) / 256), 256>>>(raw, (long long)nodes, ctx->tabA, ctx->tabB);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    if (raw) cudaFree(raw);
    if (e != cudaSuccess) {
        int rc = e == cudaErrorMemoryAllocation ? GEO_ENOMEM : GEO_ECUDA;
        geo_destroy(ctx);
        return rc;
    }
    ctx->tm.A = ctx->tabA;
    ctx->tm.B = ctx->tabB;
    ctx->tm.n1 = (int)tb->n1;
    ctx->tm.n2 = (int)tb->n2;
    ctx->tm.x1_0 = tb->x1_0;
    ctx->tm.d1 = tb->d1;
    ctx->tm.inv_d1 = 1.0 / tb->d1;
    ctx->tm.x2_0 = tb->x2_0;
    ctx->tm.d2 = tb->d2;
    ctx->tm.inv_d2 = 1.0 / tb->d2;
    *out_ctx = ctx;
    return GEO_OK;
}

int geo_create_tabulated_general(geo_ctx** out_ctx, const geo_table* tb) {
    if (!out_ctx) return GEO_EINVAL;
    *out_ctx = nullptr;
    if (!tb || !tb->tab || tb->n1 < 4 || tb->n2 < 4 || tb->n1 > 0x3fffffff || tb->n2 > 0x3fffffff) return GEO_EINVAL;
    if (!(tb->d1 > 0.0) || !(tb->d2 > 0.0) || !std::isfinite(tb->d1) || !std::isfinite(tb->d2) ||
        !std::isfinite(tb->x1_0) || !std::isfinite(tb->x2_0))
        return GEO_EINVAL;
    geo_ctx* ctx = new (std::nothrow) geo_ctx;
    if (!ctx) return GEO_ENOMEM;
    memset(ctx, 0, sizeof *ctx);
    ctx->metric = GEO_TABULATED_GENERAL;
    ctx->M = NAN;
    ctx->a = NAN;
    const size_t nodes = (size_t)tb->n1 * (size_t)tb->n2;
    double* raw = nullptr;
    cudaError_t e = cudaGetDevice(&ctx->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->counter, 2 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->tabG, nodes * kTabgStride * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&raw, kTabgFields * nodes * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(raw, tb->tab, kTabgFields * nodes * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        tabg_pack_kernel<<<(unsigned)((nodes + 255) / 256), 256>>>(raw, (long long)nodes, ctx->tabG);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
    }
    if (raw) cudaFree(raw);
    if (e != cudaSuccess) {
        int rc = e == cudaErrorMemoryAllocation ? GEO_ENOMEM : GEO_ECUDA;
        geo_destroy(ctx);
        return rc;
    }
    ctx->tgm.G = ctx->tabG;
    ctx->tgm.n1 = (int)tb->n1;
    ctx->tgm.n2 = (int)tb->n2;
    ctx->tgm.x1_0 = tb->x1_0;
    ctx->tgm.d1 = tb->d1;
    ctx->tgm.inv_d1 = 1.0 / tb->d1;
    ctx->tgm.x2_0 = tb->x2_0;
    ctx->tgm.d2 = tb->d2;
    ctx->tgm.inv_d2 = 1.0 / tb->d2;
    *out_ctx = ctx;
    return GEO_OK;
}

void geo_destroy(geo_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard guard(ctx->device);      // frees go to the ctx's device (best effort if the switch fails)
    if (ctx->tabA) cudaFree(ctx->tabA);
    if (ctx->tabB) cudaFree(ctx->tabB);
    if (ctx->tabG) cudaFree(ctx->tabG);
    for (int k = 0; k < 2; ++k)
        if (ctx->host_stream[k]) cudaStreamDestroy(ctx->host_stream[k]);
    if (ctx->scratch) cudaFree(ctx->scratch);
    if (ctx->counter) cudaFree(ctx->counter);
    delete ctx;
}

double geo_horizon_radius(const geo_ctx* ctx) {
    if (!ctx || ctx->metric == GEO_TABULATED || ctx->metric == GEO_TABULATED_GENERAL) return NAN;
    return ctx->M + std::sqrt(ctx->M * ctx->M - ctx->a * ctx->a);
}

const char* geo_last_error(const geo_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }

int geo_integrate(geo_ctx* ctx, const double* state_in, int64_t n, double h, int64_t nsteps,
                  const geo_stop* stop, int64_t snapshot_every, const geo_out* out, void* cuda_stream) {
    int rc = validate(ctx, state_in, n, h, nsteps, stop, snapshot_every, out, true);
    if (rc != GEO_OK || n == 0) return rc;
    GEO_ON_CTX_DEVICE(ctx);
    return launch(ctx, state_in, n, h, nsteps, stop, snapshot_every, out, (cudaStream_t)cuda_stream, ctx->counter);
}

}  // extern "C"

// Host-buffer pipeline shared by geo_integrate_host and geo_integrate_adaptive_host.  Small jobs: one H2D, one
// launch, one D2H.  Jobs whose buffers exceed kHostChunkBytes are cut into particle chunks that ping-pong between two
// device scratch slots on two streams, so that the D2H of chunk k (the paper's measured bottleneck)
// overlaps the kernel of chunk k+1, and the next kernel's CTAs fill the SMs the previous kernel's tail leaves idle.
// `enqueue(d_in, c, d_out, d_rejected, stream, counter)` launches the kernel for one chunk of c particles.
// Arguments are validated by the caller; the ctx's device is current.
template <class Enqueue>
static int host_pipeline(geo_ctx* ctx, const double* state_in, int64_t n, const geo_out* out, bool with_snapshots,
                         int32_t* rejected, Enqueue enqueue) {
    const size_t N = (size_t)n;
    const int ncomp = with_snapshots ? popcount8(out->snap_mask) : 0;
    const size_t snap_pp = with_snapshots ? (size_t)out->snap_capacity * ncomp * 8 : 0;   // bytes per particle
    const size_t bytes_pp = 48 + 64 + 4 + 8 + (out->eq_cross_r ? 8 : 0) + (out->health ? 8 : 0) + (out->coarse_steps ? 4 : 0) +
                            (rejected ? 4 : 0) + snap_pp + (snap_pp ? 4 : 0);
    // chunking: only when the transfers are large, never below ~2 waves of resident lanes per chunk
    const size_t kHostChunkBytes = (size_t)768 << 20;
    const size_t min_chunk = (size_t)ctx->sm_count * GEO_MIN_CTAS_PER_SM * kBlock * 2;
    size_t nchunks = (N * bytes_pp + kHostChunkBytes - 1) / kHostChunkBytes;
    if (nchunks > N / min_chunk) nchunks = N / min_chunk;
    if (nchunks < 1) nchunks = 1;
    const size_t C = ((N + nchunks - 1) / nchunks + 31) & ~(size_t)31;      // particles per chunk
    const int nslots = nchunks > 1 ? 2 : 1;

    const size_t b_in = align256(6 * C * 8), b_fin = align256(8 * C * 8), b_st = align256(C * 4),
                 b_steps = align256(C * 8), b_eq = out->eq_cross_r ? align256(C * 8) : 0,
                 b_he = out->health ? align256(C * 8) : 0, b_sn = align256(C * snap_pp),
                 b_sc = snap_pp ? align256(C * 4) : 0, b_co = out->coarse_steps ? align256(C * 4) : 0,
                 b_rej = rejected ? align256(C * 4) : 0;
    const size_t slot_bytes = b_in + b_fin + b_st + b_steps + b_eq + b_he + b_sn + b_sc + b_co + b_rej;
    const size_t total = slot_bytes * nslots;
    cudaError_t e;
    for (int k = 0; k < nslots; ++k) {
        if (!ctx->host_stream[k]) {
            e = cudaStreamCreateWithFlags(&ctx->host_stream[k], cudaStreamNonBlocking);
            if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaStreamCreate");
        }
    }
    if (total > ctx->scratch_bytes) {
        if (ctx->scratch) cudaFree(ctx->scratch);
        ctx->scratch = nullptr;
        ctx->scratch_bytes = 0;
        e = cudaMalloc(&ctx->scratch, total);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMalloc(scratch)");
        ctx->scratch_bytes = total;
    }
    // after the first enqueue every error path drains both streams before returning: no copy into the caller's
    // buffers is left in flight behind a failed call
    auto bail = [&](int code) {
        for (int k = 0; k < nslots; ++k) cudaStreamSynchronize(ctx->host_stream[k]);
        return code;
    };
    for (size_t k = 0, lo = 0; lo < N; ++k, lo += C) {
        const size_t c = N - lo < C ? N - lo : C;
        const int slot = (int)(k % nslots);
        cudaStream_t s = ctx->host_stream[slot];
        char* base = static_cast<char*>(ctx->scratch) + slot_bytes * slot;
        size_t off = 0;
        auto take = [&](size_t b) { char* q = b ? base + off : nullptr; off += b; return q; };
        double* d_in = (double*)take(b_in);
        geo_out d = *out;
        d.final_state = (double*)take(b_fin);
        d.status = (int32_t*)take(b_st);
        d.steps_done = (int64_t*)take(b_steps);
        d.eq_cross_r = (double*)take(b_eq);
        d.health = (double*)take(b_he);
        d.snapshots = (double*)take(b_sn);
        d.snap_count = (int32_t*)take(b_sc);
        d.coarse_steps = (int32_t*)take(b_co);
        int32_t* d_rej = (int32_t*)take(b_rej);
        if (!snap_pp) d.snapshots = nullptr;
        e = cudaSuccess;
        for (int q = 0; q < 6 && e == cudaSuccess; ++q)      // SoA [6][n] -> [6][c]
            e = cudaMemcpyAsync(d_in + q * c, state_in + q * N + lo, c * 8, cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) return bail(fail_cuda(ctx, e, "H2D state_in"));
        if (d.snapshots) {
            // slots >= snap_count[i] come back as NaN (all-ones pattern)
            e = cudaMemsetAsync(d.snapshots, 0xFF, c * snap_pp, s);
            if (e != cudaSuccess) return bail(fail_cuda(ctx, e, "memset snapshots"));
        }
        const int rc = enqueue(d_in, (int64_t)c, &d, d_rej, s, ctx->counter + slot);
        if (rc != GEO_OK) return bail(rc);
        for (int q = 0; q < 8 && e == cudaSuccess; ++q)      // SoA [8][c] -> [8][n]
            e = cudaMemcpyAsync(out->final_state + q * N + lo, d.final_state + q * c, c * 8, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(out->status + lo, d.status, c * 4, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(out->steps_done + lo, d.steps_done, c * 8, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d.eq_cross_r) e = cudaMemcpyAsync(out->eq_cross_r + lo, d.eq_cross_r, c * 8, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d.health) e = cudaMemcpyAsync(out->health + lo, d.health, c * 8, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d.snapshots)
            e = cudaMemcpyAsync(reinterpret_cast<char*>(out->snapshots) + lo * snap_pp, d.snapshots, c * snap_pp, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d.snap_count) e = cudaMemcpyAsync(out->snap_count + lo, d.snap_count, c * 4, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d.coarse_steps) e = cudaMemcpyAsync(out->coarse_steps + lo, d.coarse_steps, c * 4, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && d_rej) e = cudaMemcpyAsync(rejected + lo, d_rej, c * 4, cudaMemcpyDeviceToHost, s);
        if (e != cudaSuccess) return bail(fail_cuda(ctx, e, "D2H outputs"));
    }
    for (int k = 0; k < nslots; ++k) {
        e = cudaStreamSynchronize(ctx->host_stream[k]);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaStreamSynchronize");
    }
    return GEO_OK;
}

extern "C" {

int geo_integrate_host(geo_ctx* ctx, const double* state_in, int64_t n, double h, int64_t nsteps,
                       const geo_stop* stop, int64_t snapshot_every, const geo_out* out) {
    int rc = validate(ctx, state_in, n, h, nsteps, stop, snapshot_every, out, false);
    if (rc != GEO_OK || n == 0) return rc;
    GEO_ON_CTX_DEVICE(ctx);
    return host_pipeline(ctx, state_in, n, out, snapshot_every > 0, nullptr,
                         [&](const double* d_in, int64_t c, const geo_out* d, int32_t*, cudaStream_t s, unsigned long long* counter) {
                             return launch(ctx, d_in, c, h, nsteps, stop, snapshot_every, d, s, counter);
                         });
}

// Argument checks of the adaptive entry points (device and host variants).
static int validate_adaptive(geo_ctx* ctx, const double* state_in, int64_t n, const geo_adaptive* ctl, int64_t max_attempts,
                             const geo_stop* stop, const geo_out* out, const int32_t* rejected, bool check_align) {
    int rc = validate(ctx, state_in, n, 1.0, 0, stop, 0, out, check_align);
    if (rc != GEO_OK) return rc;
    if (ctx->metric == GEO_KERR_SCHILD && stop && stop->flags != 0) return fail(ctx, GEO_EINVAL, "GEO_KERR_SCHILD: the adaptive path takes no flags");
    if ((ctx->metric == GEO_TABULATED || ctx->metric == GEO_TABULATED_GENERAL) && stop && stop->flags != 0) return fail(ctx, GEO_EINVAL, "tabulated metrics: the adaptive path takes no flags");
    if (!ctl) return fail(ctx, GEO_EINVAL, "ctl must not be NULL");
    if (!std::isfinite(ctl->h0) || !(ctl->h0 > 0.0)) return fail(ctx, GEO_EINVAL, "h0 must be finite and > 0");
    if (!(ctl->rtol >= 0.0) || !(ctl->atol >= 0.0) || !(ctl->rtol + ctl->atol > 0.0) || std::isinf(ctl->atol))
        return fail(ctx, GEO_EINVAL, "rtol, atol must be >= 0, not both 0 (rtol = +inf: fixed step)");
    if (!(ctl->h_min >= 0.0) || !(ctl->tau_end > 0.0)) return fail(ctx, GEO_EINVAL, "h_min >= 0 and tau_end > 0 required");
    if (max_attempts < 0 || max_attempts > 0x7fffffffLL) return fail(ctx, GEO_EINVAL, "max_attempts must be in [0, 2^31)");
    if (stop->flags & ~GEO_FLAG_CARTESIAN_SNAP) return fail(ctx, GEO_EINVAL, "the adaptive path takes GEO_FLAG_CARTESIAN_SNAP only");
    if (!(ctl->snap_dtau >= 0.0) || std::isinf(ctl->snap_dtau)) return fail(ctx, GEO_EINVAL, "snap_dtau must be finite and >= 0");
    if (ctl->snap_dtau > 0.0 && n > 0) {
        if (!out->snapshots || !out->snap_count) return fail(ctx, GEO_EINVAL, "snap_dtau > 0 needs snapshots and snap_count");
        if (out->snap_capacity < 1 || out->snap_capacity > 0x7fffffffLL) return fail(ctx, GEO_EINVAL, "snap_capacity must be in [1, 2^31)");
        if ((out->snap_mask & 0xFFu) == 0 || (out->snap_mask & ~0xFFu)) return fail(ctx, GEO_EINVAL, "snap_mask must select 1..8 of the 8 components");
    }
    if (check_align && misaligned(rejected)) return fail(ctx, GEO_EINVAL, "device pointers must be 16-byte aligned");
    return GEO_OK;
}

// GEO_KERR_SCHILD: the adaptive kernel of geo_ks_rk45.cuh (reading K6).
static int launch_adaptive_ks(geo_ctx* ctx, const double* state_in, int64_t n, const geo_adaptive* ctl, int64_t max_attempts,
                              const geo_stop* stop, const geo_out* out, int32_t* rejected, cudaStream_t stream,
                              unsigned long long* counter) {
    KsAdaptiveParams p;
    memset(&p, 0, sizeof p);
    p.in = state_in;
    p.n = n;
    p.h0 = ctl->h0;
    p.rtol = ctl->rtol;
    p.atol = ctl->atol;
    p.h_min = ctl->h_min;
    p.tau_end = ctl->tau_end;
    p.fixed_step = std::isinf(ctl->rtol) ? 1 : 0;
    p.max_attempts = (int)max_attempts;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.rejected = rejected;
    p.counter = counter;
    const bool dense = ctl->snap_dtau > 0.0;
    p.snap_dtau = ctl->snap_dtau;
    p.snaps = dense ? out->snapshots : nullptr;
    p.snap_cap = dense ? out->snap_capacity : 0;
    p.snap_mask = dense ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = dense ? popcount8(out->snap_mask) : 0;
    p.snap_count = dense ? out->snap_count : nullptr;
    p.bh.M = ctx->M;
    p.bh.a = ctx->a;
    p.bh.a2 = ctx->a * ctx->a;
    p.bh.twoM = 2.0 * ctx->M;
    p.bh.four_a2 = 4.0 * ctx->a * ctx->a;
    typedef void (*fn_t)(const KsAdaptiveParams);
    fn_t fn = dense ? (fn_t)geo_ks_rk45_kernel<true> : (fn_t)geo_ks_rk45_kernel<false>;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, kBlock, 0);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "occupancy(ks rk45)");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    const int64_t need = (n + kBlock - 1) / kBlock, resident = (int64_t)ctx->sm_count * per_sm;
    const int grid = (int)(need < resident ? need : resident);
    e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    fn<<<grid, kBlock, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

// Enqueue the RK5(4) kernel on validated arguments (device pointers); the ctx's device is current.
static int launch_adaptive(geo_ctx* ctx, const double* state_in, int64_t n, const geo_adaptive* ctl, int64_t max_attempts,
                           const geo_stop* stop, const geo_out* out, int32_t* rejected, cudaStream_t stream,
                           unsigned long long* counter) {
    if (ctx->metric == GEO_KERR_SCHILD) return launch_adaptive_ks(ctx, state_in, n, ctl, max_attempts, stop, out, rejected, stream, counter);
    AdaptiveParams p;
    memset(&p, 0, sizeof p);
    p.in = state_in;
    p.n = n;
    p.h0 = ctl->h0;
    p.rtol = ctl->rtol;
    p.atol = ctl->atol;
    p.h_min = ctl->h_min;
    p.tau_end = ctl->tau_end;
    p.fixed_step = std::isinf(ctl->rtol) ? 1 : 0;
    p.max_attempts = (int)max_attempts;
    p.r_capture = stop->r_capture;
    p.r_escape = stop->r_escape;
    p.kappa = stop->kind == GEO_TIMELIKE ? 1.0 : 0.0;
    p.fin = out->final_state;
    p.status = out->status;
    p.steps_done = reinterpret_cast<long long*>(out->steps_done);
    p.eq_cross_r = out->eq_cross_r;
    p.health = out->health;
    p.rejected = rejected;
    p.counter = counter;
    const bool dense = ctl->snap_dtau > 0.0;
    p.snap_dtau = ctl->snap_dtau;
    p.snaps = dense ? out->snapshots : nullptr;
    p.snap_cap = dense ? out->snap_capacity : 0;
    p.snap_mask = dense ? (out->snap_mask & 0xFFu) : 0;
    p.ncomp = dense ? popcount8(out->snap_mask) : 0;
    p.cartesian = (stop->flags & GEO_FLAG_CARTESIAN_SNAP) ? 1 : 0;
    p.snap_count = dense ? out->snap_count : nullptr;
    p.bh.M = ctx->M;
    p.bh.a = ctx->a;
    p.bh.a2 = ctx->a * ctx->a;
    p.bh.twoM = 2.0 * ctx->M;
    p.bh.twoMa = 2.0 * ctx->M * ctx->a;
    fill_trig_consts(p.bh.tc);
    p.tm = ctx->tm;
    p.tgm = ctx->tgm;
    typedef void (*fn_t)(const AdaptiveParams);
    fn_t fn = ctx->metric == GEO_KERR ? (dense ? (fn_t)geo_rk45_kernel<METRIC_KERR, true> : (fn_t)geo_rk45_kernel<METRIC_KERR, false>)
            : ctx->metric == GEO_TABULATED ? (dense ? (fn_t)geo_rk45_kernel<METRIC_TAB, true> : (fn_t)geo_rk45_kernel<METRIC_TAB, false>)
            : ctx->metric == GEO_TABULATED_GENERAL ? (dense ? (fn_t)geo_rk45_kernel<METRIC_TABG, true> : (fn_t)geo_rk45_kernel<METRIC_TABG, false>)
                                           : (dense ? (fn_t)geo_rk45_kernel<METRIC_SCHW, true> : (fn_t)geo_rk45_kernel<METRIC_SCHW, false>);
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, kBlock, 0);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "occupancy(rk45)");
    if (per_sm < 1) return fail(ctx, GEO_ECUDA, "kernel does not fit on an SM");
    const int64_t need = (n + kBlock - 1) / kBlock, resident = (int64_t)ctx->sm_count * per_sm;
    const int grid = (int)(need < resident ? need : resident);
    e = cudaMemsetAsync(counter, 0, sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "cudaMemsetAsync(counter)");
    fn<<<grid, kBlock, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "kernel launch");
    return GEO_OK;
}

int geo_integrate_adaptive(geo_ctx* ctx, const double* state_in, int64_t n, const geo_adaptive* ctl,
                           int64_t max_attempts, const geo_stop* stop, const geo_out* out, int32_t* rejected,
                           void* cuda_stream) {
    int rc = validate_adaptive(ctx, state_in, n, ctl, max_attempts, stop, out, rejected, true);
    if (rc != GEO_OK || n == 0) return rc;
    GEO_ON_CTX_DEVICE(ctx);
    if (ctl->snap_dtau > 0.0 && misaligned(out->snapshots)) return fail(ctx, GEO_EINVAL, "device pointers must be 16-byte aligned");
    return launch_adaptive(ctx, state_in, n, ctl, max_attempts, stop, out, rejected, (cudaStream_t)cuda_stream, ctx->counter);
}

// Host-buffer entry point of the adaptive path: the chunked double-buffered pipeline of geo_integrate_host.
int geo_integrate_adaptive_host(geo_ctx* ctx, const double* state_in, int64_t n, const geo_adaptive* ctl,
                                int64_t max_attempts, const geo_stop* stop, const geo_out* out, int32_t* rejected) {
    int rc = validate_adaptive(ctx, state_in, n, ctl, max_attempts, stop, out, rejected, false);
    if (rc != GEO_OK || n == 0) return rc;
    GEO_ON_CTX_DEVICE(ctx);
    return host_pipeline(ctx, state_in, n, out, ctl->snap_dtau > 0.0, rejected,
                         [&](const double* d_in, int64_t c, const geo_out* d, int32_t* d_rej, cudaStream_t s, unsigned long long* counter) {
                             return launch_adaptive(ctx, d_in, c, ctl, max_attempts, stop, d, d_rej, s, counter);
                         });
}

int geo_launch_info(geo_ctx* ctx, int64_t n, int32_t flags, int64_t snapshot_every, int32_t info[4]) {
    if (!ctx || !info || n < 0) return GEO_EINVAL;
    GEO_ON_CTX_DEVICE(ctx);
    if (ctx->metric == GEO_TABULATED) {
        info[1] = kTabBlock;
        return plan_tab(ctx, n, flags, &info[0], &info[3], &info[2], snapshot_every > 0);
    }
    if (ctx->metric == GEO_TABULATED_GENERAL) {
        info[1] = tabg_block(flags);
        return plan_tabg(ctx, n, flags, &info[0], &info[3], &info[2], snapshot_every > 0);
    }
    if (ctx->metric == GEO_KERR_SCHILD) {
        info[1] = kBlock;
        return plan_ks(ctx, n, flags, snapshot_every > 0, nullptr, &info[0], &info[3], &info[2]);
    }
    LaunchPlan lp;
    int rc = plan_launch(ctx, n, flags, snapshot_every, 8, &lp);
    if (rc != GEO_OK) return rc;
    info[0] = lp.grid;
    info[1] = lp.block;
    info[2] = lp.regs;
    info[3] = lp.ctas_per_sm;
    return GEO_OK;
}

int geo_probe_dfma(geo_ctx* ctx, int64_t iters, double* sink, double* n_fma, void* cuda_stream) {
    if (!ctx || !sink || !n_fma || iters < 1) return GEO_EINVAL;
    GEO_ON_CTX_DEVICE(ctx);
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)dfma_probe_kernel, 256, 0);
    if (e != cudaSuccess) return fail_cuda(ctx, e, "occupancy(dfma_probe)");
    const int grid = ctx->sm_count * per_sm;
    dfma_probe_kernel<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(iters, sink);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(ctx, e, "dfma_probe launch");
    *n_fma = (double)grid * 256.0 * 64.0 * (double)iters;
    return GEO_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// geo_integrate_host_noalloc (include/geo.h): the geo_integrate_host operation for callers that cannot allocate.
// All device scratch -- the work-queue head of the persistent kernel and the staging of inputs and outputs -- is the
// file-scope array below: fixed offsets for GEO_NOALLOC_MAX_N particles, 256-byte aligned, held by every device that
// loads this module until the process exits.  In HOST code `g_noalloc_scratch` is only a handle of the symbol, not a
// device address: the address is resolved once per device by cudaGetSymbolAddress (noalloc_device) and that pointer is
// what the kernel gets.
namespace {
constexpr size_t kNaN = GEO_NOALLOC_MAX_N;
constexpr size_t kNaHead = 0;                          // unsigned long long work-queue head (256 B reserved)
constexpr size_t kNaIn = 256;                          // [6][n] double
constexpr size_t kNaFin = kNaIn + 48 * kNaN;           // [8][n] double
constexpr size_t kNaSteps = kNaFin + 64 * kNaN;        // [n] int64
constexpr size_t kNaEq = kNaSteps + 8 * kNaN;          // [n] double
constexpr size_t kNaHealth = kNaEq + 8 * kNaN;         // [n] double
constexpr size_t kNaStatus = kNaHealth + 8 * kNaN;     // [n] int32
constexpr size_t kNaCoarse = kNaStatus + 4 * kNaN;     // [n] int32
constexpr size_t kNaBytes = kNaCoarse + 4 * kNaN;      // 256 + 144 * 65536 = 9 437 440
static_assert(kNaBytes == 256 + 144 * kNaN, "scratch size stated in geo.h");
static_assert(kNaN % 64 == 0, "every sub-buffer starts on a 256-byte boundary");
}  // namespace

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNaBytes];

namespace {
constexpr int kNaMaxDevices = 64;
struct NoallocDevice {
    unsigned char* base;   // device address of g_noalloc_scratch on this device
    int sm_count;
    bool ready;
};
NoallocDevice g_na_dev[kNaMaxDevices];
std::mutex g_na_mutex;                 // serialises the calls of one process: they share the scratch
thread_local char g_na_err[256] = "";

int na_fail(int code, const char* msg) {
    snprintf(g_na_err, sizeof g_na_err, "%s", msg);
    return code;
}
int na_fail_cuda(cudaError_t e, const char* what) {
    snprintf(g_na_err, sizeof g_na_err, "%s: %s", what, cudaGetErrorString(e));
    return GEO_ECUDA;
}

// Set-up, once per device, with that device current (the caller holds g_na_mutex).
int noalloc_device(int device, NoallocDevice** out) {
    if (device < 0 || device >= kNaMaxDevices) return na_fail(GEO_EINVAL, "device ordinal beyond the per-device table of the allocation-free path");
    NoallocDevice& d = g_na_dev[device];
    if (!d.ready) {
        unsigned char* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_scratch);
        if (e != cudaSuccess) return na_fail_cuda(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) return na_fail(GEO_ECUDA, "static scratch is not 256-byte aligned");
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return na_fail_cuda(e, "cudaDeviceGetAttribute(SM count)");
        d.base = ptr;
        d.sm_count = sms;
        d.ready = true;
    }
    *out = &d;
    return GEO_OK;
}
}  // namespace

extern "C" {

const char* geo_noalloc_last_error(void) { return g_na_err; }

int geo_integrate_host_noalloc(int metric, double M, double a, const double* state_in, int64_t n, double h,
                               int64_t nsteps, const geo_stop* stop, const geo_out* out, void* cuda_stream) {
    g_na_err[0] = 0;
    if (metric != GEO_SCHWARZSCHILD && metric != GEO_KERR) return na_fail(GEO_EINVAL, "metric must be GEO_SCHWARZSCHILD or GEO_KERR");
    if (!(M > 0.0) || !std::isfinite(M) || !(std::fabs(a) <= M)) return na_fail(GEO_EINVAL, "M > 0 and |a| <= M required");
    if (metric == GEO_SCHWARZSCHILD && a != 0.0) return na_fail(GEO_EINVAL, "Schwarzschild requires a == 0");
    // a ctx on the stack: no device memory of its own, its queue head is the first word of the static scratch
    geo_ctx local;
    memset(&local, 0, sizeof local);
    local.metric = metric;
    local.M = M;
    local.a = a;
    int rc = validate(&local, state_in, n, h, nsteps, stop, 0, out, false);
    if (rc != GEO_OK) return na_fail(rc, local.err);
    if (stop->flags & ~(GEO_FLAG_PLAIN_UPDATE | GEO_FLAG_STATIC_MAP)) return na_fail(GEO_EINVAL, "the allocation-free path takes GEO_FLAG_PLAIN_UPDATE and GEO_FLAG_STATIC_MAP only");
    if (n > (int64_t)kNaN) {
        snprintf(g_na_err, sizeof g_na_err, "n = %lld exceeds GEO_NOALLOC_MAX_N = %lld (size of the static device scratch)", (long long)n, (long long)kNaN);
        return GEO_EINVAL;
    }
    if (n == 0) return GEO_OK;

    std::lock_guard<std::mutex> lock(g_na_mutex);
    cudaError_t e = cudaGetDevice(&local.device);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaGetDevice");
    NoallocDevice* dev = nullptr;
    rc = noalloc_device(local.device, &dev);
    if (rc != GEO_OK) return rc;
    local.sm_count = dev->sm_count;

    cudaStream_t s = (cudaStream_t)cuda_stream;
    unsigned char* base = dev->base;
    const size_t N = (size_t)n;
    double* d_in = reinterpret_cast<double*>(base + kNaIn);
    geo_out d;
    memset(&d, 0, sizeof d);
    d.final_state = reinterpret_cast<double*>(base + kNaFin);
    d.status = reinterpret_cast<int32_t*>(base + kNaStatus);
    d.steps_done = reinterpret_cast<int64_t*>(base + kNaSteps);
    d.eq_cross_r = out->eq_cross_r ? reinterpret_cast<double*>(base + kNaEq) : nullptr;
    d.health = out->health ? reinterpret_cast<double*>(base + kNaHealth) : nullptr;
    d.coarse_steps = out->coarse_steps ? reinterpret_cast<int32_t*>(base + kNaCoarse) : nullptr;

    // after the first enqueue every error path drains the stream: no copy into the caller's buffers stays in flight
    auto bail = [&](int code) {
        cudaStreamSynchronize(s);
        return code;
    };
    e = cudaMemcpyAsync(d_in, state_in, 6 * N * 8, cudaMemcpyHostToDevice, s);      // SoA [6][n], contiguous on both sides
    if (e != cudaSuccess) return bail(na_fail_cuda(e, "H2D state_in"));
    // launch() clears the queue head (scratch + kNaHead) on the stream, then starts the same kernel geo_integrate_host runs
    rc = launch(&local, d_in, n, h, nsteps, stop, 0, &d, s, reinterpret_cast<unsigned long long*>(base + kNaHead));
    if (rc != GEO_OK) return bail(na_fail(rc, local.err));
    e = cudaMemcpyAsync(out->final_state, d.final_state, 8 * N * 8, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out->status, d.status, N * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out->steps_done, d.steps_done, N * 8, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess && d.eq_cross_r) e = cudaMemcpyAsync(out->eq_cross_r, d.eq_cross_r, N * 8, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess && d.health) e = cudaMemcpyAsync(out->health, d.health, N * 8, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess && d.coarse_steps) e = cudaMemcpyAsync(out->coarse_steps, d.coarse_steps, N * 4, cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) return bail(na_fail_cuda(e, "D2H outputs"));
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return na_fail_cuda(e, "cudaStreamSynchronize");
    return GEO_OK;
}

}  // extern "C"
