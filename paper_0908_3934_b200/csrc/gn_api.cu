// gn_api.cu -- host logic of the C ABI declared in include/gn.h: validation, workspace layout,
// uploads, step sequencing and read-back.  No arithmetic of the method runs here; every step of
// the path is a kernel in gn_kernels.cu.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "gn_internal.h"

namespace {

thread_local char g_create_error[256] = "";

struct Layout {
    size_t V, W, r, p2, hm, hh, c, acc, bias, refr, cls, ring, row, tgt, wfx, dly, counters, q_count;
    size_t s_edge, s_dly, min_dly, q_seg, spk_log;
    size_t w_f32, perm, ls_hist, pl_list, csc_off, csc_edge, csc_src, w_stage;
    size_t raster, trace, scratch_row64, scratch_abs, scratch_pos, scratch_net, scratch_chk, total;
};

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int check_config(const gn_config *cfg, char *err, size_t errn)
{
    auto fail = [&](const char *m) { snprintf(err, errn, "%s", m); return GN_E_INVALID_ARG; };
    if (!cfg) return fail("cfg is NULL");
    if (cfg->n_vertices == 0 || cfg->n_vertices > 0xFFFFFF00u) return fail("n_vertices must be in [1, 2^32-256]");
    if (cfg->dim != 2 && cfg->dim != 3) return fail("dim must be 2 or 3");
    if (cfg->n_edges >= 0xFFFFFFFFull) return fail("n_edges must be < 2^32 - 1");
    if (cfg->ring_slots < 2 || cfg->ring_slots > 255) return fail("ring_slots must be in [2, 255]");
    if (cfg->n_classes < 1 || cfg->n_classes > GN_MAX_CLASSES) return fail("n_classes must be in [1, GN_MAX_CLASSES]");
    if (!(cfg->dt_ms > 0.0f)) return fail("dt_ms must be > 0");
    if (cfg->n_networks < 1 || cfg->n_networks > cfg->n_vertices) return fail("n_networks must be in [1, n_vertices]");
    if (cfg->obs_stride > 0 && cfg->trace_capacity_frames == 0) return fail("obs_stride > 0 needs trace_capacity_frames > 0");
    if (cfg->obs_stride > 0 && !(cfg->tau_ca_ms > 0.0f)) return fail("obs_stride > 0 needs tau_ca_ms > 0");
    if (cfg->delivery_mode > GN_DELIVER_RING_STEPWISE) return fail("delivery_mode must be GN_DELIVER_AUTO, _RING, _QUEUE, _RESIDENT or _RING_STEPWISE");
    if (cfg->stdp_alpha != 0.0f) {
        if (!(cfg->stdp_beta >= 0.0f) || !isfinite(cfg->stdp_alpha) || !isfinite(cfg->stdp_beta)) return fail("stdp_alpha must be finite and stdp_beta finite and >= 0");
        if (cfg->delivery_mode != GN_DELIVER_AUTO && cfg->delivery_mode != GN_DELIVER_RING)
            return fail("plastic weights (stdp_alpha != 0) need delivery_mode GN_DELIVER_AUTO or GN_DELIVER_RING");
    }
    const uint32_t qg = cfg->queue_group;
    if (qg != 0 && (qg > 16 || (qg & (qg - 1)) != 0)) return fail("queue_group must be 0 or a power of two in 1..16");
    return GN_OK;
}

// Groups beyond the current one whose events the update kernel delivers itself (GnDev::q_window).
static const uint32_t kQueueWindow = 2u;

// Resolved delivery plan of queue mode: log2(slots per group), groups per lap, log arrays, spikes per step the log holds.
struct QueuePlan {
    bool on;
    uint32_t q_log, q_nb, arrays;
    uint32_t log_cap;
};

QueuePlan make_plan(const gn_config *cfg)
{
    const uint64_t N = cfg->n_vertices, Npad = (N + 127) / 128 * 128, E = cfg->n_edges, D = cfg->ring_slots;
    QueuePlan q{};
    uint32_t group = cfg->queue_group ? cfg->queue_group : 8u;
    while (group > 1 && D % group != 0) group >>= 1;      // the ring depth must be a whole number of groups
    q.on = cfg->delivery_mode == GN_DELIVER_QUEUE ||
           (cfg->delivery_mode == GN_DELIVER_AUTO && D >= 32 && D * Npad * 4 > (48ull << 20));
    if (E == 0 || cfg->stdp_alpha != 0.0f) q.on = false;    // plastic weights: delivery at arrival time (gn_arrive_kernel)
    q.q_log = 0;
    while ((1u << q.q_log) < group) q.q_log++;
    q.q_nb = (uint32_t)(D / group);
    q.arrays = q.q_nb > kQueueWindow ? q.q_nb - kQueueWindow + 1u : 0u;   // boundaries of group offsets W+1 .. nb (+ the row's end)
    uint64_t cap = cfg->queue_capacity ? cfg->queue_capacity : (N + 15) / 16;
    if (cfg->queue_capacity == 0 && cap < 1024) cap = 1024;
    if (cap > Npad) cap = Npad;                           // a step has at most N spikes
    if (cap > (1ull << 23)) cap = 1ull << 23;             // 255 steps x log_cap entries are indexed in 32 bits
    q.log_cap = (uint32_t)((cap + 31) / 32 * 32);
    return q;
}

Layout make_layout(const gn_config *cfg)
{
    const size_t N = cfg->n_vertices, Npad = (N + 127) / 128 * 128, E = cfg->n_edges, D = cfg->ring_slots;
    const bool obs = cfg->obs_stride > 0;
    Layout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    L.V = take(Npad * 4); L.W = take(Npad * 4); L.r = take(Npad * 4); L.p2 = take(Npad * 4);
    L.hm = take(Npad * 4); L.hh = take(Npad * 4);
    L.c = take(obs ? Npad * 4 : 0); L.acc = take(obs ? Npad * 4 : 0);
    L.bias = take(Npad * 4);
    L.refr = take(Npad); L.cls = take(Npad);
    L.ring = take(D * Npad * 4);
    L.row = take((Npad + 1) * 4); L.tgt = take(E * 4); L.wfx = take(E * 4); L.dly = take(E);
    L.counters = take(32);
    const QueuePlan qp = make_plan(cfg);
    L.q_count = take(256 * 8);       // +0: the persistent step driver's barrier counter; +64: spikes logged per step slot
                                     // (at most 255 x 4 bytes); +1536: the two GN_FAULTS counters
    {
        size_t rows = cfg->raster_capacity_steps, need_rows = qp.on ? (size_t)(kQueueWindow + 1u) << qp.q_log : 2;
        if (cfg->stdp_alpha != 0.0f) need_rows = D;     // plastic mode: the raster is the spikes in flight
        if (rows < need_rows) rows = need_rows;
        L.raster = take(rows * (Npad / 32) * 4);
    }
    L.trace = take(obs ? (size_t)cfg->trace_capacity_frames * Npad * 4 : 0);
    L.min_dly = take(Npad);
    L.s_edge = take(E * 8); L.s_dly = take(E);   // every row again, sorted by delay
    const bool plastic = cfg->stdp_alpha != 0.0f;
    L.q_seg = take(qp.on || plastic ? N * D * 2 : 0);
    L.w_f32 = take(plastic ? E * 4 : 0); L.perm = take(plastic ? E * 4 : 0); L.w_stage = take(plastic ? E * 4 : 0);
    L.ls_hist = take(plastic ? (D + 1) * Npad * 4 : 0); L.pl_list = take(plastic ? D * Npad * 4 : 0);
    L.csc_off = take(plastic ? (Npad + 2) * 4 : 0); L.csc_edge = take(plastic ? E * 4 : 0); L.csc_src = take(plastic ? E * 4 : 0);
    L.spk_log = take(qp.on && qp.arrays >= 2 ? D * qp.arrays * (size_t)qp.log_cap * 4 : 0);
    L.scratch_row64 = take((N + 1) * 8); L.scratch_abs = take(N * 8);
    L.scratch_pos = take(N * cfg->dim * 4); L.scratch_net = take(((size_t)cfg->n_networks + 1) * 4);
    L.scratch_chk = take(sizeof(GnCheck));
    L.total = off;
    return L;
}

}  // namespace

struct gn_net {
    int device;          // CUDA device of the workspace: every entry point runs with it current (DeviceGuard)
    gn_config cfg;
    GnDev dev;
    Layout lay;
    cudaStream_t stream;
    uint8_t *ws;
    uint64_t t;          // steps enqueued so far
    uint64_t t_origin;   // first step simulated by this handle (0, or the t a checkpoint was restored at)
    unsigned long long sync_base;   // persistent step driver: value of its barrier counter when the next launch starts
    uint64_t routed_upto; // queue mode: steps < routed_upto have been entered into the spike log
    uint64_t zeroed_upto;  // queue mode: the log's spike counts of steps < zeroed_upto (not logged yet) are zero already
    uint64_t flushed_upto; // queue mode: every event of steps < flushed_upto is in the ring already (a read-back expanded them)
    // delivery of step t overlaps the update of step t+1 (see gn_step): side streams and their fences
    cudaStream_t s_deliver;
    cudaEvent_t ev_update, ev_deliver[2], ev_fold[4];
    bool fences_pending;
    bool has_bias;
    unsigned long long faults_seen[2];   // GN_FAULTS as last read to the host (plastic mode): non-zero stops gn_step
    unsigned long long barrier_broken;   // grid_sync[1] as last read: the persistent driver's barrier timed out
    unsigned long long *scratch_abs;     // N x 8 bytes of the workspace, free after gn_create (per-target sums of |w_fx|)
    // measuring mode (gn_profile)
    bool profile;
    std::vector<cudaEvent_t> ev;      // pool, reused chunk after chunk
    std::vector<uint8_t> ev_kind;     // kernel that runs between event i and event i+1 (0xFF = none)
    size_t ev_used;
    double prof_ms[4];
    uint64_t prof_n[4];
    uint8_t prof_last;               // kind of the launch after the last event
    uint64_t launches;                // every kernel launched by gn_step since gn_create
    char err[256];
};

namespace {

int set_err(gn_net *net, int code, const char *fmt, ...)
{
    char *dst = net ? net->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 256, fmt, ap);
    va_end(ap);
    return code;
}

// Makes `device` current for the lifetime of the guard and restores the caller's device afterwards: a handle works
// from any thread whatever device is current there (multi-replica hosts).
struct DeviceGuard {
    int prev = -1, want;
    explicit DeviceGuard(int device) : want(device)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != want) cudaSetDevice(want);
    }
    ~DeviceGuard()
    {
        if (prev >= 0 && prev != want) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

#define GN_CUDA(net, call)                                                                        \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return set_err(net, GN_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_));        \
    } while (0)

}  // namespace

// Records the message gn_last_error(NULL) returns on this thread and hands the code back: for entry points that live in
// other files of the library and have no handle (gn_static.cu).
int gn_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_create_error, sizeof g_create_error, fmt, ap);
    va_end(ap);
    return code;
}

extern "C" {

int gn_query_workspace(const gn_config *cfg, size_t *bytes)
{
    if (!bytes) { snprintf(g_create_error, sizeof g_create_error, "bytes is NULL"); return GN_E_INVALID_ARG; }
    int rc = check_config(cfg, g_create_error, sizeof g_create_error);
    if (rc) return rc;
    *bytes = make_layout(cfg).total;
    return GN_OK;
}

int gn_create(const gn_config *cfg, const gn_class_params *classes, const float *positions,
              const uint64_t *row_offsets, const uint32_t *targets, const float *weights,
              const uint8_t *delays, const uint8_t *vertex_class, const float *bias,
              const uint32_t *net_offsets, void *workspace, size_t workspace_bytes,
              void *cuda_stream, gn_net **out)
{
    if (out) *out = nullptr;
    int rc = check_config(cfg, g_create_error, sizeof g_create_error);
    if (rc) return rc;
    if (!out || !classes || !row_offsets || !vertex_class || !workspace)
        return set_err(nullptr, GN_E_INVALID_ARG, "NULL argument (out/classes/row_offsets/vertex_class/workspace)");
    if (cfg->n_edges && (!targets || !weights))
        return set_err(nullptr, GN_E_INVALID_ARG, "targets/weights are NULL with n_edges > 0");
    if (cfg->n_edges && !delays && !positions)
        return set_err(nullptr, GN_E_INVALID_ARG, "need delays or positions");
    if (!delays && !(cfg->speed > 0.0f))
        return set_err(nullptr, GN_E_INVALID_ARG, "speed must be > 0 when delays == NULL");
    if (cfg->n_networks > 1 && !net_offsets)
        return set_err(nullptr, GN_E_INVALID_ARG, "n_networks > 1 needs net_offsets");
    if (((uintptr_t)workspace & 255u) != 0)
        return set_err(nullptr, GN_E_INVALID_ARG, "workspace must be 256-byte aligned");
    const Layout L = make_layout(cfg);
    if (workspace_bytes < L.total)
        return set_err(nullptr, GN_E_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, need %zu", workspace_bytes, L.total);

    int n_dev = 0;
    GN_CUDA(nullptr, cudaGetDeviceCount(&n_dev));
    if (n_dev < 1) return set_err(nullptr, GN_E_CUDA, "no CUDA device");
    cudaPointerAttributes attr{};
    GN_CUDA(nullptr, cudaPointerGetAttributes(&attr, workspace));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return set_err(nullptr, GN_E_INVALID_ARG, "workspace is not device memory");

    DeviceGuard guard(attr.device);           // the workspace's device, whatever is current in this thread
    gn_net *net = new (std::nothrow) gn_net();
    if (!net) return set_err(nullptr, GN_E_INVALID_ARG, "out of host memory");
    net->device = attr.device;
    net->cfg = *cfg;
    net->lay = L;
    net->stream = (cudaStream_t)cuda_stream;
    net->ws = (uint8_t *)workspace;
    net->t = 0;
    net->t_origin = 0;
    net->routed_upto = 0;
    net->flushed_upto = 0;
    net->zeroed_upto = 0;
    net->sync_base = 0;
    net->s_deliver = nullptr;
    net->ev_update = net->ev_deliver[0] = net->ev_deliver[1] = net->ev_fold[0] = net->ev_fold[1] = net->ev_fold[2] = net->ev_fold[3] = nullptr;
    net->fences_pending = false;
    net->has_bias = bias != nullptr;
    net->profile = false;
    net->prof_last = 0xFF;
    net->ev_used = 0;
    net->launches = 0;
    for (int k = 0; k < 4; ++k) { net->prof_ms[k] = 0.0; net->prof_n[k] = 0; }
    net->err[0] = 0;

    const uint32_t N = cfg->n_vertices, Npad = (N + 127) / 128 * 128;
    const uint64_t E = cfg->n_edges;
    uint8_t *ws = net->ws;
    GnDev &d = net->dev;
    memset(&d, 0, sizeof d);
    d.N = N; d.Npad = Npad; d.D = cfg->ring_slots; d.words_pad = Npad / 32; d.n_classes = cfg->n_classes;
    d.obs_stride = cfg->obs_stride; d.raster_cap = cfg->raster_capacity_steps;
    d.trace_cap = cfg->obs_stride ? cfg->trace_capacity_frames : 0;
    d.seed_lo = (uint32_t)cfg->seed; d.seed_hi = (uint32_t)(cfg->seed >> 32);
    d.dt = cfg->dt_ms;
    // constants: computed once in double, rounded once
    d.keep_c = cfg->obs_stride ? (float)(1.0 - (double)cfg->dt_ms / (double)cfg->tau_ca_ms) : 0.0f;
    d.ca_jump = cfg->ca_jump;
    d.obs_gain = cfg->obs_gain; d.obs_offset = cfg->obs_offset; d.obs_sigma = cfg->obs_sigma;
    d.inv_stride = cfg->obs_stride ? (float)(1.0 / (double)cfg->obs_stride) : 0.0f;
    d.V = (float *)(ws + L.V); d.W = (float *)(ws + L.W); d.r = (float *)(ws + L.r); d.p2 = (float *)(ws + L.p2);
    d.hm = (float *)(ws + L.hm); d.hh = (float *)(ws + L.hh);
    d.c = cfg->obs_stride ? (float *)(ws + L.c) : nullptr;
    d.acc = cfg->obs_stride ? (float *)(ws + L.acc) : nullptr;
    d.bias = (float *)(ws + L.bias);
    d.refr = ws + L.refr; d.cls = ws + L.cls;
    d.ring = (int32_t *)(ws + L.ring);
    d.row = (uint32_t *)(ws + L.row); d.tgt = (uint32_t *)(ws + L.tgt);
    d.wfx = (int32_t *)(ws + L.wfx); d.dly = ws + L.dly;
    d.counters = (unsigned long long *)(ws + L.counters);
    d.raster = (uint32_t *)(ws + L.raster);
    const QueuePlan qp = make_plan(cfg);
    d.raster_rows = cfg->raster_capacity_steps;   // the delivery kernels read the spike lists of up to two groups
    {
        uint32_t need_rows = qp.on ? (kQueueWindow + 1u) << qp.q_log : 2u;
        if (cfg->stdp_alpha != 0.0f) need_rows = cfg->ring_slots;
        if (d.raster_rows < need_rows) d.raster_rows = need_rows;
    }
    d.queue_mode = qp.on ? 1u : 0u;
    d.q_log = qp.q_log; d.q_nb = qp.q_nb; d.q_arrays = qp.arrays; d.log_cap = qp.log_cap;
    d.grid_sync = (unsigned long long *)(ws + L.q_count);
    d.log_n = (uint32_t *)(ws + L.q_count + 64);
    d.faults = (unsigned long long *)(ws + L.q_count + 1536);
    d.s_edge = (uint2 *)(ws + L.s_edge); d.s_dly = ws + L.s_dly; d.min_dly = ws + L.min_dly;
    d.packed = Npad <= (1u << 24) ? 1u : 0u;
    d.q_window = kQueueWindow;
    if (qp.on) {
        d.q_seg = (uint16_t *)(ws + L.q_seg);
        d.spk_log = (uint32_t *)(ws + L.spk_log);
    }
    if (cfg->stdp_alpha != 0.0f) {       // plastic weights: per-delay boundaries = the segment table with groups of one slot
        d.plastic = 1u;
        d.stdp_dta = (float)((double)cfg->dt_ms * (double)cfg->stdp_alpha);
        d.stdp_beta = cfg->stdp_beta;
        d.q_log = 0u; d.q_nb = cfg->ring_slots; d.q_arrays = 0u;
        d.q_seg = (uint16_t *)(ws + L.q_seg);
        d.w_f32 = (float *)(ws + L.w_f32); d.perm = (uint32_t *)(ws + L.perm); d.w_stage = (float *)(ws + L.w_stage);
        d.ls_hist = (int32_t *)(ws + L.ls_hist); d.pl_list = (uint32_t *)(ws + L.pl_list);
        d.csc_off = (uint32_t *)(ws + L.csc_off); d.csc_edge = (uint32_t *)(ws + L.csc_edge); d.csc_src = (uint32_t *)(ws + L.csc_src);
    }
    d.trace = cfg->obs_stride ? (float *)(ws + L.trace) : nullptr;
    for (uint32_t k = 0; k < cfg->n_classes; ++k) {
        const gn_class_params &c = classes[k];
        GnClassDev &q = d.cls_tab[k];
        q.a = c.a; q.b = c.b; q.c_reset = c.c_reset; q.d = c.d;
        q.k2 = c.k2; q.k1 = c.k1; q.k0 = c.k0; q.v_peak = c.v_peak;
        q.direct = !(c.tau_syn_ms > 0.0f);
        q.keep_s = q.direct ? 0.0f : (float)(1.0 - (double)cfg->dt_ms / (double)c.tau_syn_ms);
        q.alpha = (!q.direct && c.psc_alpha != 0.0f) ? 1u : 0u;       // alpha-function PSC, a = 1/tau_syn
        q.a2 = q.alpha ? (float)(1.0 / ((double)c.tau_syn_ms * (double)c.tau_syn_ms)) : 0.0f;
        q.two_a = q.alpha ? (float)(2.0 / (double)c.tau_syn_ms) : 0.0f;
        if (q.alpha) d.any_alpha = 1u;
        if (c.model != 0.0f && c.model != 1.0f) {
            delete net;
            return set_err(nullptr, GN_E_INVALID_ARG, "class %u: model must be 0 (Izhikevich) or 1 (Hodgkin-Huxley)", k);
        }
        q.hh = c.model == 1.0f ? 1u : 0u;
        if (q.hh) {            // Hodgkin-Huxley constants: formed once in double, rounded once
            const float *rate[6] = {c.hh_am, c.hh_bm, c.hh_ah, c.hh_bh, c.hh_an, c.hh_bn};
            bool ok = c.hh_c > 0.0f;
            for (int f = 0; f < 6; ++f) ok = ok && rate[f][2] != 0.0f && isfinite(rate[f][0]) && isfinite(rate[f][1]) && isfinite(rate[f][2]);
            if (!ok) {
                delete net;
                return set_err(nullptr, GN_E_INVALID_ARG, "class %u (Hodgkin-Huxley): hh_c must be > 0 and every rate function needs finite {A, V_half, k} with k != 0", k);
            }
            d.any_hh = 1u;
            q.hh_dt_c = (float)((double)cfg->dt_ms / (double)c.hh_c);
            q.hh_g_na = c.hh_g_na; q.hh_g_k = c.hh_g_k; q.hh_g_l = c.hh_g_l;
            q.hh_e_na = c.hh_e_na; q.hh_e_k = c.hh_e_k; q.hh_e_l = c.hh_e_l;
            double val[6];     // the rates at hh_v_rest, for the gates' initial steady states alpha / (alpha + beta)
            for (int f = 0; f < 6; ++f) {
                const double A = rate[f][0], vh = rate[f][1], kk = rate[f][2], u = ((double)c.hh_v_rest - vh) * (1.0 / kk);
                const bool linoid = f == 0 || f == 4, sigmoid = f == 3;
                q.hh_ak[f] = (float)(linoid ? A * kk : A);
                q.hh_vh[f] = rate[f][1];
                q.hh_inv_k[f] = (float)(1.0 / kk);
                val[f] = linoid ? (A * kk) * (fabs(u) < 0.05 ? fma(u, fma(u, 1.0 / 12.0, 0.5), 1.0) : u / (1.0 - exp(-u)))
                       : sigmoid ? A / (1.0 + exp(-u)) : A * exp(-u);
            }
            q.hh_v0 = c.hh_v_rest;
            q.hh_m0 = (float)(val[0] / (val[0] + val[1]));
            q.hh_h0 = (float)(val[2] / (val[2] + val[3]));
            q.hh_n0 = (float)(val[4] / (val[4] + val[5]));
        }
        const double R = nearbyint((double)c.refractory_ms / (double)cfg->dt_ms);
        if (!(R >= 0.0) || R > 255.0) {
            delete net;
            return set_err(nullptr, GN_E_INVALID_ARG, "class %u: refractory_ms / dt_ms must round to 0..255 steps", k);
        }
        q.R = (uint32_t)R;
        const double pthr = (((double)c.drive_rate_hz * (double)cfg->dt_ms) * 1e-3) * 4294967296.0;
        q.drive_thr = !(pthr > 0.0) ? 0u : (pthr >= 4294967295.0 ? 4294967295u : (uint32_t)floor(pthr));
        const double kick = nearbyint((double)c.drive_kick * 65536.0);
        if (!(fabs(kick) < 2147483648.0)) {
            delete net;
            return set_err(nullptr, GN_E_INVALID_ARG, "class %u: drive_kick out of the fixed-point range", k);
        }
        q.kick_fx = (int32_t)kick;
        if (q.drive_thr) d.any_drive = 1u;
    }

    cudaStream_t st = net->stream;
    uint64_t *row64 = (uint64_t *)(ws + L.scratch_row64);
    unsigned long long *abs_in = (unsigned long long *)(ws + L.scratch_abs);
    net->scratch_abs = abs_in;
    float *pos_d = (float *)(ws + L.scratch_pos);
    uint32_t *net_d = (uint32_t *)(ws + L.scratch_net);
    GnCheck *chk_d = (GnCheck *)(ws + L.scratch_chk);

#define GN_CREATE_CUDA(call)                                                                      \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) {                                                                  \
            cudaStreamSynchronize(st);   /* copies from caller buffers may still be in flight */  \
            delete net;                                                                           \
            return set_err(nullptr, GN_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_));    \
        }                                                                                         \
    } while (0)

    // zero everything the step loop accumulates into or reads before writing
    GN_CREATE_CUDA(cudaMemsetAsync(ws, 0, L.tgt, st));                       // state, bias, refr, cls, ring, row
    GN_CREATE_CUDA(cudaMemsetAsync(ws + L.counters, 0, L.min_dly - L.counters, st));   // counters, bucket counts, raster, trace
    GN_CREATE_CUDA(cudaMemsetAsync(abs_in, 0, (size_t)N * 8, st));
    GN_CREATE_CUDA(cudaMemsetAsync(chk_d, 0, sizeof(GnCheck), st));
    // uploads (host or device sources)
    GN_CREATE_CUDA(cudaMemcpyAsync(row64, row_offsets, ((size_t)N + 1) * 8, cudaMemcpyDefault, st));
    GN_CREATE_CUDA(cudaMemcpyAsync(d.cls, vertex_class, N, cudaMemcpyDefault, st));
    if (E) {
        GN_CREATE_CUDA(cudaMemcpyAsync(d.tgt, targets, E * 4, cudaMemcpyDefault, st));
        GN_CREATE_CUDA(cudaMemcpyAsync(d.wfx, weights, E * 4, cudaMemcpyDefault, st));   // fp32 bits, quantised in place
        if (delays) GN_CREATE_CUDA(cudaMemcpyAsync(d.dly, delays, E, cudaMemcpyDefault, st));
        else GN_CREATE_CUDA(cudaMemcpyAsync(pos_d, positions, (size_t)N * cfg->dim * 4, cudaMemcpyDefault, st));
    }
    if (bias) GN_CREATE_CUDA(cudaMemcpyAsync(d.bias, bias, (size_t)N * 4, cudaMemcpyDefault, st));
    if (net_offsets)
        GN_CREATE_CUDA(cudaMemcpyAsync(net_d, net_offsets, ((size_t)cfg->n_networks + 1) * 4, cudaMemcpyDefault, st));
    // device-side conversion and validation
    GN_CREATE_CUDA(gnk_convert_rows(d, row64, E, chk_d, st));
    GN_CREATE_CUDA(gnk_init_state(d, chk_d, st));
    GnCheck chk{};
    GN_CREATE_CUDA(cudaMemcpyAsync(&chk, chk_d, sizeof chk, cudaMemcpyDeviceToHost, st));
    GN_CREATE_CUDA(cudaStreamSynchronize(st));
    if (chk.bad_row || chk.bad_class) {
        delete net;
        return set_err(nullptr, GN_E_BAD_GRAPH, chk.bad_row ? "row_offsets: not monotone, row_offsets[0] != 0 or row_offsets[N] != n_edges"
                                                            : "vertex_class: id >= n_classes");
    }
    // the (small) network table: checked on the host, read back from the device copy so device-resident inputs work too
    std::vector<uint32_t> net_h((size_t)cfg->n_networks + 1);
    if (net_offsets) {
        GN_CREATE_CUDA(cudaMemcpyAsync(net_h.data(), net_d, net_h.size() * 4, cudaMemcpyDeviceToHost, st));
        GN_CREATE_CUDA(cudaStreamSynchronize(st));
    } else {
        net_h[0] = 0; net_h[1] = N;
        GN_CREATE_CUDA(cudaMemcpyAsync(net_d, net_h.data(), 8, cudaMemcpyHostToDevice, st));
        GN_CREATE_CUDA(cudaStreamSynchronize(st));
    }
    uint32_t max_net = 0;
    {
        bool ok = net_h.front() == 0 && net_h.back() == N;
        for (size_t b = 0; ok && b + 1 < net_h.size(); ++b) {
            if (net_h[b + 1] < net_h[b]) ok = false;
            else if (net_h[b + 1] - net_h[b] > max_net) max_net = net_h[b + 1] - net_h[b];
        }
        if (!ok) {
            delete net;
            return set_err(nullptr, GN_E_BAD_GRAPH, "net_offsets must start at 0, end at n_vertices and never decrease");
        }
    }
    // resident mode: every network in one CTA -- or one thread-block cluster of up to 16 CTAs x 1,024 vertices --
    // with its ring in shared memory (gn_resident_kernel)
    {
        const uint32_t cluster = max_net <= 1024 ? 1u : (max_net + 1023u) / 1024u;
        const uint32_t threads = cluster > 1 ? 1024u : (max_net <= 32 ? 32u : (max_net + 31u) / 32u * 32u);
        const size_t smem = (size_t)cfg->ring_slots * threads * 4 + (size_t)4 * (threads / 4 + 2) * 16;
        bool fits = cluster <= 16 && smem <= 200u * 1024u;
        if (fits && cluster > 1) {
            GnDev probe = d;
            probe.res_cluster = cluster; probe.res_threads = threads; probe.res_smem = (uint32_t)smem;
            probe.n_networks = cfg->n_networks; probe.packed = Npad <= (1u << 24) ? 1u : 0u;
            GN_CREATE_CUDA(gnk_resident_cluster_ok(probe, &fits));
        }
        if (cfg->delivery_mode == GN_DELIVER_RESIDENT && !fits) {
            delete net;
            return set_err(nullptr, GN_E_INVALID_ARG, "GN_DELIVER_RESIDENT needs every network to have <= 16,384 vertices and the ring "
                                                      "of 1,024 vertices (ring_slots x 1,024 x 4 bytes) to fit 200 KB of shared memory");
        }
        d.n_networks = cfg->n_networks;
        d.net_off = net_d;
        if (fits && !d.plastic && (cfg->delivery_mode == GN_DELIVER_RESIDENT || cfg->delivery_mode == GN_DELIVER_AUTO)) {
            d.resident = 1u;
            d.res_cluster = cluster;
            d.res_threads = threads;
            d.res_smem = (uint32_t)smem;
            d.queue_mode = 0u;
        }
    }
    // ring mode on a small network: one kernel per step (the update delivers), bound by launch latency not work
    d.fused = (!d.resident && !d.queue_mode && !d.plastic && Npad <= (1u << 18)) ? 1u : 0u;
    // ... and when its whole update grid can be co-resident, one cooperative launch per gn_step call (gn_persist_kernel).
    // (GN_DELIVER_RING_STEPWISE keeps the per-step path: measurements and tests of it.)
    if (d.fused && cfg->delivery_mode != GN_DELIVER_RING_STEPWISE) {
        bool ok = false;
        GN_CREATE_CUDA(gnk_persist_ok(d, &ok));
        d.persist = ok ? 1u : 0u;
    }
    if (E) {
        GN_CREATE_CUDA(gnk_quantise(d, E, chk_d, st));
        if (!delays) GN_CREATE_CUDA(gnk_delays_from_positions(d, pos_d, cfg->dim, cfg->speed, chk_d, st));
        GN_CREATE_CUDA(gnk_validate(d, net_offsets ? net_d : nullptr, cfg->n_networks, abs_in, chk_d, st));
    }
    GN_CREATE_CUDA(gnk_check_overflow(d, abs_in, chk_d, st));
    GN_CREATE_CUDA(cudaMemsetAsync(d.min_dly, 0xFF, Npad, st));
    if (E) GN_CREATE_CUDA(gnk_sort_rows(d, chk_d, st));
    if (d.plastic) {                     // in-edge lists (scratch: the per-target sums, no longer needed), no spike yet
        GN_CREATE_CUDA(cudaMemsetAsync(d.csc_off, 0, ((size_t)Npad + 2) * 4, st));
        GN_CREATE_CUDA(cudaMemsetAsync(abs_in, 0, (size_t)N * 4, st));
        GN_CREATE_CUDA(gnk_build_csc(d, E, (uint32_t *)abs_in, st));
        GN_CREATE_CUDA(cudaMemsetAsync(d.ls_hist, 0xFF, ((size_t)cfg->ring_slots + 1) * Npad * 4, st));
    }
    GN_CREATE_CUDA(cudaMemcpyAsync(&chk, chk_d, sizeof chk, cudaMemcpyDeviceToHost, st));
    GN_CREATE_CUDA(cudaStreamSynchronize(st));
#undef GN_CREATE_CUDA
    if (chk.bad_target || chk.bad_delay || chk.cross_net || chk.bad_weight || chk.bad_position) {
        delete net;
        return set_err(nullptr, GN_E_BAD_GRAPH, "%s",
                       chk.bad_target ? "targets: id >= n_vertices"
                       : chk.bad_position ? "positions: NaN or infinite coordinate on an edge (eq. 25 has no delay for it)"
                       : chk.bad_delay ? "delay outside [1, ring_slots-1]"
                       : chk.cross_net ? "edge crosses two networks"
                                       : "weight is NaN or outside the int32 fixed-point range");
    }
    if (chk.overflow) {
        delete net;
        return set_err(nullptr, GN_E_OVERFLOW_RISK, "some target's sum |w_fx| + |kick_fx| exceeds 2^31 - 1");
    }
    // side stream: the delivery kernel (ring mode: of step t; queue mode: of a slot group) runs beside later updates
    {
        int lo = 0, hi = 0;
        cudaError_t e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&net->s_deliver, cudaStreamNonBlocking, hi);
        cudaEvent_t *evs[7] = {&net->ev_update, &net->ev_deliver[0], &net->ev_deliver[1], &net->ev_fold[0], &net->ev_fold[1],
                               &net->ev_fold[2], &net->ev_fold[3]};
        for (int k = 0; k < 7 && e == cudaSuccess; ++k) e = cudaEventCreateWithFlags(evs[k], cudaEventDisableTiming);
        if (e != cudaSuccess) {
            gn_destroy(net);
            return set_err(nullptr, GN_E_CUDA, "creating side streams failed: %s", cudaGetErrorString(e));
        }
    }
    *out = net;
    return GN_OK;
}

// ---- measuring mode: one event wherever the KIND of kernel changes (a run of consecutive launches of one kernel
// is timed as a whole, so an event's own cost is not charged to every launch), collected every kProfChunk steps ----
static const size_t kProfChunk = 256;

static int prof_mark(gn_net *net, uint8_t kind_after)
{
    if (kind_after <= 3) net->prof_n[kind_after] += 1;                  // every launch is counted ...
    if (kind_after == net->prof_last && kind_after != 0xFF) return GN_OK;   // ... but only a change of kind is marked
    net->prof_last = kind_after;
    if (net->ev_used == net->ev.size()) {
        cudaEvent_t e;
        GN_CUDA(net, cudaEventCreate(&e));
        net->ev.push_back(e);
        net->ev_kind.push_back(0xFF);
    }
    GN_CUDA(net, cudaEventRecord(net->ev[net->ev_used], net->stream));
    net->ev_kind[net->ev_used] = kind_after;
    net->ev_used++;
    return GN_OK;
}

static int prof_collect(gn_net *net)
{
    if (net->ev_used == 0) return GN_OK;
    GN_CUDA(net, cudaStreamSynchronize(net->stream));
    for (size_t i = 0; i + 1 < net->ev_used; ++i) {
        const uint8_t k = net->ev_kind[i];
        if (k > 3) continue;
        float ms = 0.f;
        GN_CUDA(net, cudaEventElapsedTime(&ms, net->ev[i], net->ev[i + 1]));
        net->prof_ms[k] += (double)ms;
    }
    net->ev_used = 0;
    net->prof_last = 0xFF;
    return GN_OK;
}

// Make the caller's stream wait for everything the side streams still have in flight.
static int join_streams(gn_net *net)
{
    if (!net->fences_pending) return GN_OK;
    GN_CUDA(net, cudaStreamWaitEvent(net->stream, net->ev_deliver[0], 0));
    GN_CUDA(net, cudaStreamWaitEvent(net->stream, net->ev_deliver[1], 0));
    for (int k = 0; k < 4; ++k) GN_CUDA(net, cudaStreamWaitEvent(net->stream, net->ev_fold[k], 0));
    net->fences_pending = false;
    return GN_OK;
}

// Ring mode.  One step t is  update(t) -> deliver(t).  update(t) needs update(t-1) and deliver(t-2): events
// with delay 1 are sent by update(t-1) itself, so the earliest slot deliver(t-1) writes is t+1, and deliver(t)
// runs on a side stream beside update(t+1).
//
// Queue mode.  Steps come in groups of G = 2^q_log (the ring rows of one group are folded together); W = q_window.
// update(t), t in group h, sends every event due in groups h .. h+W-1 itself.  After the last update of group h two
// kernels go to the side stream, beside the updates of group h+1 (and beside each other):
//   gn_log_kernel sends the events of group h's spikes due in group h+W and enters the spikes into the spike log;
//   gn_fold_kernel expands, out of the log of groups h+W-nb .. h-1 (complete since the previous launches on that
//   stream), the events due in group h+W into that group's ring rows.
// update(first step of h+W) waits for that launch: W-1 groups of slack.  The raster rows a launch reads are
// overwritten W+1 groups later, after the next launches on the side stream.
// In profiling mode everything runs on the caller's stream in that order, so per-kernel times are clean.
static int zero_log_counts(gn_net *net, uint64_t t0, uint64_t t1, cudaStream_t st)
{
    const GnDev &d = net->dev;
    const uint32_t s0 = (uint32_t)(t0 % d.D), n = (uint32_t)(t1 - t0);
    const uint32_t first = n < d.D - s0 ? n : d.D - s0;
    GN_CUDA(net, cudaMemsetAsync(d.log_n + s0, 0, (size_t)first * 4, st));
    if (first < n) GN_CUDA(net, cudaMemsetAsync(d.log_n, 0, (size_t)(n - first) * 4, st));
    return GN_OK;
}

// Logs the steps not yet logged (all inside one group) and, when g_fold != ~0, folds slot group g_fold out of the log.
static int route_pending(gn_net *net, cudaStream_t st, bool prof, uint64_t g_fold)
{
    const GnDev &d = net->dev;
    if (!d.queue_mode) return GN_OK;
    const uint32_t n_batch = (uint32_t)(net->t - net->routed_upto);
    uint64_t t_win = 0;
    uint32_t n_win = 0;
    if (g_fold != ~0ull && d.q_arrays >= 2u) {          // steps of groups g-nb .. g-W-1 that no read-back has expanded yet
        const uint64_t lo_g = g_fold >= d.q_nb ? g_fold - d.q_nb : 0ull;
        const uint64_t hi = g_fold >= d.q_window ? (g_fold - d.q_window) << d.q_log : 0ull;
        uint64_t lo = lo_g << d.q_log;
        if (lo < net->flushed_upto) lo = net->flushed_upto;
        const uint64_t hi_c = hi < net->routed_upto ? hi : net->routed_upto;
        if (hi_c > lo) { t_win = lo; n_win = (uint32_t)(hi_c - lo); }
    }
    if (n_batch == 0 && n_win == 0) return GN_OK;
    int rc;
    if (n_batch) {
        const uint64_t z0 = net->routed_upto > net->zeroed_upto ? net->routed_upto : net->zeroed_upto;
        if (z0 < net->t && (rc = zero_log_counts(net, z0, net->t, st))) return rc;      // (steady state: the previous launch did it)
        // at a group's end the next group's counts are zeroed by this launch: what they hold now -- the counts of the group a lap
        // earlier -- was last wanted by the fold of the next group itself, issued a launch ago (or clipped away by a read-back)
        const uint32_t G = 1u << d.q_log;
        const bool at_group_end = (net->t & (uint64_t)(G - 1u)) == 0;
        const uint32_t zero_next = (at_group_end && d.D >= 2u * G) ? G : 0u;
        if (prof && (rc = prof_mark(net, 1))) return rc;
        GN_CUDA(net, gnk_log(d, net->routed_upto, n_batch, zero_next, st));
        if (net->zeroed_upto < net->t + zero_next) net->zeroed_upto = net->t + zero_next;
        net->launches++;
    }
    if (n_win) {
        if (prof && (rc = prof_mark(net, 3))) return rc;
        GN_CUDA(net, gnk_fold(d, t_win, n_win, g_fold, n_batch != 0 && !prof, st));
        net->launches++;
    }
    net->routed_upto = net->t;
    return GN_OK;
}

int gn_step(gn_net *net, uint64_t n_steps)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    const GnDev &d = net->dev;
    const uint32_t G = 1u << d.q_log;
    if (d.resident) {      // the whole call is one launch (or a few, so that a kept raster window is never lapped)
        const bool raster_on = d.raster_cap > 0;
        uint64_t left = n_steps;
        while (left) {
            uint64_t n = left > 0x40000000ull ? 0x40000000ull : left;
            if (raster_on && n > d.raster_rows) n = d.raster_rows;
            int rc;
            if (net->profile && (rc = prof_mark(net, 0))) return rc;
            GN_CUDA(net, gnk_resident(d, net->t, (uint32_t)n, net->has_bias, raster_on, net->stream));
            net->launches++;
            net->t += n;
            left -= n;
        }
        if (net->profile) {
            int rc = prof_mark(net, 0xFF);
            return rc ? rc : prof_collect(net);
        }
        return GN_OK;
    }
    if (d.plastic) {       // plastic weights: arrivals of step t, the update, then eq. 33 and eq. 32, all on the caller's stream
        if (net->faults_seen[0] || net->faults_seen[1])
            return set_err(net, GN_E_OVERFLOW_RISK, "the plastic weights outgrew the fixed-point ring (GN_FAULTS: %llu deliveries of a weight outside "
                           "+-32768, %llu targets whose sum of |w| no longer fits int32): stepping is refused",
                           net->faults_seen[0], net->faults_seen[1]);
        for (uint64_t s = 0; s < n_steps; ++s) {
            const uint64_t t = net->t;
            const bool prof = net->profile;
            int rc;
            if (prof && (rc = prof_mark(net, 1))) return rc;
            GN_CUDA(net, gnk_arrive(d, t, net->t_origin, net->stream));
            if (prof && (rc = prof_mark(net, 0))) return rc;
            GN_CUDA(net, gnk_update(d, t, net->has_bias, net->stream));
            if (prof && (rc = prof_mark(net, 3))) return rc;
            GN_CUDA(net, gnk_plasticity(d, t, net->t_origin, net->stream));
            net->launches += 4;
            net->t = t + 1;
            if (d.obs_stride && (t + 1) % d.obs_stride == 0) {      // a5 reads the calcium state only: nothing in it depends on the weights
                if (prof && (rc = prof_mark(net, 2))) return rc;
                GN_CUDA(net, gnk_observe(d, (t + 1) / d.obs_stride - 1, net->stream));
                net->launches++;
            }
            if (prof && (s + 1) % kProfChunk == 0 && ((rc = prof_mark(net, 0xFF)) || (rc = prof_collect(net)))) return rc;
        }
        if (net->profile) {
            int rc = prof_mark(net, 0xFF);
            return rc ? rc : prof_collect(net);
        }
        return GN_OK;
    }
    if (d.persist) {       // ring mode, co-resident grid: the whole call is one cooperative launch
        if (net->barrier_broken)
            return set_err(net, GN_E_CUDA, "the persistent step driver's grid barrier timed out: the results of this handle are invalid");
        uint64_t left = n_steps;
        while (left) {
            const uint64_t n = left > 0x40000000ull ? 0x40000000ull : left;
            int rc;
            if (net->profile && (rc = prof_mark(net, 0))) return rc;
            GN_CUDA(net, gnk_persist(d, net->t, (uint32_t)n, net->has_bias, d.grid_sync, &net->sync_base, net->stream));
            net->launches++;
            net->t += n;
            left -= n;
        }
        if (net->profile) {
            int rc = prof_mark(net, 0xFF);
            return rc ? rc : prof_collect(net);
        }
        return GN_OK;
    }
    for (uint64_t s = 0; s < n_steps; ++s) {
        const uint64_t t = net->t;
        const bool prof = net->profile;
        cudaStream_t s_upd = net->stream;
        cudaStream_t s_del = prof ? net->stream : net->s_deliver;
        int rc;
        if (!prof) {
            if (d.queue_mode) {
                if (t % G == 0) GN_CUDA(net, cudaStreamWaitEvent(s_upd, net->ev_fold[(t / G) & 3ull], 0));   // fold of this group
            } else if (t >= 2) {
                GN_CUDA(net, cudaStreamWaitEvent(s_upd, net->ev_deliver[t & 1ull], 0));                          // deliver(t-2)
            }
        }
        if (prof && (rc = prof_mark(net, 0))) return rc;
        GN_CUDA(net, gnk_update(d, t, net->has_bias, s_upd));
        net->launches++;
        net->t = t + 1;
        const bool group_end = d.queue_mode && (t % G == G - 1u);
        if (!prof && !d.fused && (!d.queue_mode || group_end)) {
            GN_CUDA(net, cudaEventRecord(net->ev_update, s_upd));
            GN_CUDA(net, cudaStreamWaitEvent(s_del, net->ev_update, 0));
        }
        if (d.fused) {
            // the update kernel delivered everything itself
        } else if (!d.queue_mode) {
            if (prof && (rc = prof_mark(net, 1))) return rc;  // also counts the step's spikes: runs even with E = 0
            GN_CUDA(net, gnk_deliver(d, t, s_del));
            net->launches++;
            if (!prof) GN_CUDA(net, cudaEventRecord(net->ev_deliver[t & 1ull], s_del));
            net->fences_pending = !prof;
        } else if (group_end) {
            if ((rc = route_pending(net, s_del, prof, t / G + d.q_window))) return rc;
            if (!prof) GN_CUDA(net, cudaEventRecord(net->ev_fold[(t / G + d.q_window) & 3ull], s_del));
            net->fences_pending = !prof;
        }
        if (d.obs_stride && (t + 1) % d.obs_stride == 0) {
            if (prof && (rc = prof_mark(net, 2))) return rc;
            GN_CUDA(net, gnk_observe(d, (t + 1) / d.obs_stride - 1, s_upd));
            net->launches++;
        }
        if (prof && (s + 1) % kProfChunk == 0 && ((rc = prof_mark(net, 0xFF)) || (rc = prof_collect(net)))) return rc;
    }
    if (net->profile) {
        int rc = prof_mark(net, 0xFF);
        return rc ? rc : prof_collect(net);
    }
    return join_streams(net);
}

// Spikes and delivered events are counted once their step is logged, and logged events reach the ring only when their
// slot group is folded: readers of counters and ring call this.  fold_too: every event of every completed step goes
// into the ring now (what direct delivery would hold), and the log is marked consumed up to here.
static int flush_delivery(gn_net *net, bool fold_too)
{
    const GnDev &d = net->dev;
    int rc = join_streams(net);
    if (rc) return rc;
    if ((rc = route_pending(net, net->stream, false, ~0ull))) return rc;
    if (fold_too && d.queue_mode && d.q_arrays >= 2u && net->flushed_upto < net->t) {
        // groups up to (h-1)+W were folded by the regular launches (h = group of the next step); the later ones, as far
        // as a logged event can reach (nb groups ahead), are folded here for the steps done so far
        const uint64_t h = net->t >> d.q_log;
        for (uint64_t g = h + d.q_window; g <= h + d.q_nb; ++g)
            if ((rc = route_pending(net, net->stream, false, g))) return rc;
        net->flushed_upto = net->t;
    }
    return GN_OK;
}

int gn_profile(gn_net *net, int enable)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    int rc = join_streams(net);
    if (rc) return rc;
    net->profile = enable != 0;
    if (enable) {
        for (int k = 0; k < 4; ++k) { net->prof_ms[k] = 0.0; net->prof_n[k] = 0; }
        net->ev_used = 0;
    }
    return GN_OK;
}

int gn_profile_read(gn_net *net, double ms[4], uint64_t launches[5])
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    if (!ms || !launches) return set_err(net, GN_E_INVALID_ARG, "NULL output");
    for (int k = 0; k < 4; ++k) { ms[k] = net->prof_ms[k]; launches[k] = net->prof_n[k]; }
    launches[4] = net->launches;
    return GN_OK;
}

static int copy_out(gn_net *net, void *dst, const void *src, size_t bytes, int dst_is_device)
{
    GN_CUDA(net, cudaMemcpyAsync(dst, src, bytes, dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, net->stream));
    if (!dst_is_device) GN_CUDA(net, cudaStreamSynchronize(net->stream));
    return GN_OK;
}

int gn_read_state(gn_net *net, int which, void *dst, size_t dst_bytes, int dst_is_device)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    if (!dst) return set_err(net, GN_E_INVALID_ARG, "dst is NULL");
    const GnDev &d = net->dev;
    const size_t N = d.N, E = net->cfg.n_edges;
    const void *src = nullptr;
    size_t need = 0;
    switch (which) {
    case GN_V: src = d.V; need = N * 4; break;
    case GN_W: src = d.W; need = N * 4; break;
    case GN_R: src = d.r; need = N * 4; break;
    case GN_P: src = d.p2; need = N * 4; break;
    case GN_M: src = d.hm; need = N * 4; break;
    case GN_H: src = d.hh; need = N * 4; break;
    case GN_CA:
        if (!d.c) return set_err(net, GN_E_INVALID_ARG, "calcium is not maintained when obs_stride == 0");
        src = d.c; need = N * 4; break;
    case GN_REFR: src = d.refr; need = N; break;
    case GN_BIAS:
        if (!net->has_bias) return set_err(net, GN_E_INVALID_ARG, "no bias set");
        src = d.bias; need = N * 4; break;
    case GN_ACC:
        if (!d.acc) return set_err(net, GN_E_INVALID_ARG, "no frame accumulator when obs_stride == 0");
        src = d.acc; need = N * 4; break;
    case GN_RING: need = (size_t)d.D * N * 4; break;
    case GN_STEP: src = d.counters; need = 8; break;
    case GN_COUNTERS: {
        int rc = flush_delivery(net, false);
        if (rc) return rc;
        src = d.counters; need = 32; break;
    }
    case GN_FAULTS: src = d.faults; need = 16; break;
    case GN_DRIVER: {
        if (dst_bytes < 4) return set_err(net, GN_E_INVALID_ARG, "dst has %zu bytes, need 4", dst_bytes);
        const uint32_t drv = d.plastic ? GN_DRIVER_PLASTIC : d.resident ? GN_DRIVER_RESIDENT : d.queue_mode ? GN_DRIVER_QUEUE
                           : d.persist ? GN_DRIVER_PERSISTENT : d.fused ? GN_DRIVER_FUSED : GN_DRIVER_RING;
        if (!dst_is_device) { memcpy(dst, &drv, 4); return GN_OK; }
        GN_CUDA(net, cudaMemcpyAsync(dst, &drv, 4, cudaMemcpyHostToDevice, net->stream));   // pageable source: staged before the call returns
        return GN_OK;
    }
    case GN_DELAYS: src = d.dly; need = E; break;
    case GN_WEIGHTS_FX: src = d.wfx; need = E * 4; break;
    case GN_WEIGHTS:
        if (!d.plastic) return set_err(net, GN_E_INVALID_ARG, "GN_WEIGHTS is the evolving weights of a plastic network (stdp_alpha != 0); static ones are GN_WEIGHTS_FX");
        src = d.w_stage; need = E * 4; break;
    default: return set_err(net, GN_E_INVALID_ARG, "unknown state id %d", which);
    }
    if (dst_bytes < need) return set_err(net, GN_E_INVALID_ARG, "dst has %zu bytes, need %zu", dst_bytes, need);
    if (need == 0) return GN_OK;
    if (which == GN_WEIGHTS) GN_CUDA(net, gnk_weights_out(d, E, net->stream));     // back to the caller's edge order
    if (which == GN_RING) {   // internal rows are Npad wide; the caller's are N wide
        int rc = flush_delivery(net, true);
        if (rc) return rc;
        GN_CUDA(net, cudaMemcpy2DAsync(dst, N * 4, d.ring, (size_t)d.Npad * 4, N * 4, d.D,
                                       dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, net->stream));
        if (!dst_is_device) GN_CUDA(net, cudaStreamSynchronize(net->stream));
        return GN_OK;
    }
    if (d.plastic && (which == GN_FAULTS || which == GN_WEIGHTS))      // gn_create's bound over the weights as they are now
        GN_CUDA(net, gnk_plastic_headroom(d, E, net->scratch_abs, net->stream));
    if (d.persist && !dst_is_device && (which == GN_COUNTERS || which == GN_STEP)) {
        // the persistent step driver's barrier gave up waiting (gn_persist_kernel): nothing since then can be trusted
        GN_CUDA(net, cudaMemcpyAsync(&net->barrier_broken, d.grid_sync + 1, 8, cudaMemcpyDeviceToHost, net->stream));
        GN_CUDA(net, cudaStreamSynchronize(net->stream));
        if (net->barrier_broken)
            return set_err(net, GN_E_CUDA, "the persistent step driver's grid barrier timed out: the results of this handle are invalid");
    }
    if (d.plastic && !dst_is_device && (which == GN_FAULTS || which == GN_COUNTERS || which == GN_WEIGHTS)) {
        // these reads wait for the stream anyway: the host learns of a fault here, and gn_step refuses to go on after one
        GN_CUDA(net, cudaMemcpyAsync(net->faults_seen, d.faults, 16, cudaMemcpyDeviceToHost, net->stream));
    }
    return copy_out(net, dst, src, need, dst_is_device);
}

int gn_write_state(gn_net *net, int which, const void *src, size_t src_bytes, int src_is_device)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    if (!src) return set_err(net, GN_E_INVALID_ARG, "src is NULL");
    const GnDev &d = net->dev;
    const size_t N = d.N;
    void *dst = nullptr;
    size_t need = N * 4;
    switch (which) {
    case GN_V: dst = d.V; break;
    case GN_W: dst = d.W; break;
    case GN_R: dst = d.r; break;
    case GN_P: dst = d.p2; break;
    case GN_M: dst = d.hm; break;
    case GN_H: dst = d.hh; break;
    case GN_CA:
        if (!d.c) return set_err(net, GN_E_INVALID_ARG, "calcium is not maintained when obs_stride == 0");
        dst = d.c; break;
    case GN_REFR: dst = d.refr; need = N; break;
    case GN_BIAS: dst = d.bias; break;
    case GN_ACC:
        if (!d.acc) return set_err(net, GN_E_INVALID_ARG, "no frame accumulator when obs_stride == 0");
        dst = d.acc; break;
    case GN_RING: need = (size_t)d.D * N * 4; break;
    case GN_STEP: need = 8; break;
    case GN_COUNTERS: need = 32; break;
    default: return set_err(net, GN_E_INVALID_ARG, "state id %d is not writable", which);
    }
    if (src_bytes < need) return set_err(net, GN_E_INVALID_ARG, "src has %zu bytes, need %zu", src_bytes, need);
    if (d.plastic && (which == GN_RING || which == GN_STEP || which == GN_COUNTERS))
        return set_err(net, GN_E_INVALID_ARG, "a plastic network (stdp_alpha != 0) cannot be restored from a checkpoint: its spikes in flight are its raster history");
    if (which == GN_RING || which == GN_STEP || which == GN_COUNTERS) {      // checkpoint / restore
        int rc = flush_delivery(net, true);       // queue mode: every pending record goes into the ring first, buckets end empty
        if (rc) return rc;
        const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        if (which == GN_RING) {                   // caller rows are N wide, internal rows Npad wide
            GN_CUDA(net, cudaMemcpy2DAsync(d.ring, (size_t)d.Npad * 4, src, N * 4, N * 4, d.D, kind, net->stream));
            GN_CUDA(net, cudaStreamSynchronize(net->stream));
            return GN_OK;
        }
        // GN_STEP: the number of completed steps t (uint64) -- the generator index, ring slot and frame phase follow from
        // it; GN_COUNTERS: all four counters (its first word is t as well).  The raster / trace windows start empty at t.
        unsigned long long c[4] = {0, 0, 0, 0};
        GN_CUDA(net, cudaMemcpyAsync(c, src, need, src_is_device ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost, net->stream));
        GN_CUDA(net, cudaStreamSynchronize(net->stream));
        if (which == GN_STEP) GN_CUDA(net, cudaMemcpyAsync(d.counters, c, 8, cudaMemcpyHostToDevice, net->stream));
        else GN_CUDA(net, cudaMemcpyAsync(d.counters, c, 32, cudaMemcpyHostToDevice, net->stream));
        GN_CUDA(net, cudaStreamSynchronize(net->stream));
        net->t = c[0];
        net->routed_upto = c[0];
        net->flushed_upto = c[0];
        net->zeroed_upto = 0;
        net->t_origin = c[0];
        return GN_OK;
    }
    GN_CUDA(net, cudaMemcpyAsync(dst, src, need, src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, net->stream));
    if (!src_is_device) GN_CUDA(net, cudaStreamSynchronize(net->stream));
    if (which == GN_BIAS) net->has_bias = true;
    return GN_OK;
}

// Rows [i0, i0+n) of a circular device window of `cap` rows, `pitch_src` bytes apart, into a dense
// destination of `width` bytes per row.
static int copy_window(gn_net *net, void *dst, const uint8_t *base, size_t pitch_src, size_t width, uint64_t cap,
                       uint64_t i0, uint64_t n, int dst_is_device)
{
    const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    uint64_t done = 0;
    while (done < n) {
        const uint64_t r0 = (i0 + done) % cap;
        const uint64_t chunk = (n - done < cap - r0) ? n - done : cap - r0;
        GN_CUDA(net, cudaMemcpy2DAsync((uint8_t *)dst + done * width, width, base + r0 * pitch_src, pitch_src, width,
                                       chunk, kind, net->stream));
        done += chunk;
    }
    if (!dst_is_device) GN_CUDA(net, cudaStreamSynchronize(net->stream));
    return GN_OK;
}

int gn_read_raster(gn_net *net, uint64_t t0, uint64_t n_steps, uint32_t *bits, size_t dst_bytes, int dst_is_device)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    const GnDev &d = net->dev;
    const size_t words = ((size_t)d.N + 31) / 32;
    if (n_steps == 0) return GN_OK;
    if (!bits) return set_err(net, GN_E_INVALID_ARG, "bits is NULL");
    if (dst_bytes < n_steps * words * 4) return set_err(net, GN_E_INVALID_ARG, "dst has %zu bytes, need %zu", dst_bytes, (size_t)(n_steps * words * 4));
    if (t0 + n_steps > net->t || d.raster_cap == 0 || t0 + d.raster_cap < net->t || t0 < net->t_origin)
        return set_err(net, GN_E_RANGE_EVICTED, "raster steps [%llu, %llu) not held: simulated %llu, window %u",
                       (unsigned long long)t0, (unsigned long long)(t0 + n_steps), (unsigned long long)net->t, d.raster_cap);
    return copy_window(net, bits, (const uint8_t *)d.raster, (size_t)d.words_pad * 4, words * 4, d.raster_rows, t0, n_steps, dst_is_device);
}

int gn_observe(gn_net *net, uint64_t frame0, uint64_t n_frames, float *trace, size_t dst_bytes, int dst_is_device)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    const GnDev &d = net->dev;
    if (!d.obs_stride) return set_err(net, GN_E_INVALID_ARG, "observation is off (obs_stride == 0)");
    if (n_frames == 0) return GN_OK;
    if (!trace) return set_err(net, GN_E_INVALID_ARG, "trace is NULL");
    const uint64_t have = net->t / d.obs_stride;
    if (dst_bytes < n_frames * d.N * 4) return set_err(net, GN_E_INVALID_ARG, "dst has %zu bytes, need %zu", dst_bytes, (size_t)(n_frames * d.N * 4));
    if (frame0 + n_frames > have || frame0 + d.trace_cap < have || frame0 < net->t_origin / d.obs_stride)
        return set_err(net, GN_E_RANGE_EVICTED, "frames [%llu, %llu) not held: emitted %llu, window %u",
                       (unsigned long long)frame0, (unsigned long long)(frame0 + n_frames), (unsigned long long)have, d.trace_cap);
    return copy_window(net, trace, (const uint8_t *)d.trace, (size_t)d.Npad * 4, (size_t)d.N * 4, d.trace_cap, frame0, n_frames, dst_is_device);
}

int gn_debug_words(void *cuda_stream, uint64_t seed, uint32_t stream_id, uint64_t idx, uint32_t first_vertex,
                   uint32_t n, uint32_t *out)
{
    if (!out && n) return set_err(nullptr, GN_E_INVALID_ARG, "out is NULL");
    GN_CUDA(nullptr, gnk_debug_words(seed, stream_id, idx, first_vertex, n, out, (cudaStream_t)cuda_stream));
    return GN_OK;
}

int gn_debug_ceilings(void *cuda_stream, void *scratch, size_t scratch_bytes, uint32_t segment_edges, double out[2])
{
    if (!scratch || !out) return set_err(nullptr, GN_E_INVALID_ARG, "NULL argument");
    cudaPointerAttributes attr{};
    GN_CUDA(nullptr, cudaPointerGetAttributes(&attr, scratch));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return set_err(nullptr, GN_E_INVALID_ARG, "scratch is not device memory");
    if (scratch_bytes < (320u << 20) || segment_edges == 0) return set_err(nullptr, GN_E_INVALID_ARG, "scratch must hold at least 320 MB and segment_edges be > 0");
    DeviceGuard guard(attr.device);
    GN_CUDA(nullptr, gnk_ceilings(scratch, scratch_bytes, segment_edges, out, (cudaStream_t)cuda_stream));
    return GN_OK;
}

int gn_debug_stream_ceilings(void *cuda_stream, void *scratch, size_t scratch_bytes, double out[2])
{
    if (!scratch || !out) return set_err(nullptr, GN_E_INVALID_ARG, "NULL argument");
    cudaPointerAttributes attr{};
    GN_CUDA(nullptr, cudaPointerGetAttributes(&attr, scratch));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return set_err(nullptr, GN_E_INVALID_ARG, "scratch is not device memory");
    if (scratch_bytes < (1024u << 20)) return set_err(nullptr, GN_E_INVALID_ARG, "scratch must hold at least 1 GB");
    DeviceGuard guard(attr.device);
    GN_CUDA(nullptr, gnk_stream_ceilings(scratch, scratch_bytes, out, (cudaStream_t)cuda_stream));
    return GN_OK;
}

const char *gn_last_error(const gn_net *net) { return net ? net->err : g_create_error; }

int gn_destroy(gn_net *net)
{
    if (!net) return GN_E_INVALID_ARG;
    DeviceGuard guard(net->device);
    if (net->s_deliver) cudaStreamSynchronize(net->s_deliver);
    cudaError_t e = cudaStreamSynchronize(net->stream);
    for (cudaEvent_t ev : net->ev) cudaEventDestroy(ev);
    cudaEvent_t evs[7] = {net->ev_update, net->ev_deliver[0], net->ev_deliver[1], net->ev_fold[0], net->ev_fold[1], net->ev_fold[2], net->ev_fold[3]};
    for (cudaEvent_t ev : evs) if (ev) cudaEventDestroy(ev);
    if (net->s_deliver) cudaStreamDestroy(net->s_deliver);
    delete net;
    return e == cudaSuccess ? GN_OK : GN_E_CUDA;
}

}  // extern "C"
