// gn_internal.h -- device-side view of one network and the kernel launchers (sm_100a only).
// Shared by gn_api.cu (host logic of the C ABI) and gn_kernels.cu (every step of the hot path).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gn.h"

// Per-class constants, derived once on the host in double and rounded once (DESIGN.md
// "Arithmetic contract"); kClassWords words each, staged into shared memory by the update kernel.
struct GnClassDev {
    float a, b, c_reset, d;
    float k2, k1, k0, v_peak;
    float keep_s;        // (float)(1 - dt/tau_s)
    uint32_t direct;     // tau_syn_ms <= 0
    uint32_t R;          // refractory steps, round(refractory_ms / dt)
    uint32_t drive_thr;  // floor(rate * dt * 1e-3 * 2^32)
    int32_t kick_fx;     // rint(kick * 2^16)
    uint32_t alpha;      // alpha-function PSC (eq. 27, 29, 30) instead of the exponential one
    float a2, two_a;     // (float)(1/tau_s^2), (float)(2/tau_s)
    uint32_t hh;         // Hodgkin-Huxley class (gn_class_params.model == 1)
    // Hodgkin-Huxley constants, each formed once in double on the host and rounded once:
    float hh_dt_c;       // dt / C
    float hh_g_na, hh_g_k, hh_g_l, hh_e_na, hh_e_k, hh_e_l;
    float hh_ak[6];      // A of each rate function (A k for the two linoid ones): alpha_m, beta_m, alpha_h, beta_h, alpha_n, beta_n
    float hh_vh[6];      // V_half
    float hh_inv_k[6];   // 1 / k
    float hh_v0, hh_m0, hh_h0, hh_n0;   // initial state: hh_v_rest and the gates' steady states there
    uint32_t pad_;
    // kClassWords is odd on purpose: a 16-byte-aligned table invites 128-bit shared-memory loads of whole rows, which
    // costs the 32-register update kernel four live registers per vertex
};
constexpr uint32_t kClassWords = 47;
static_assert(sizeof(GnClassDev) == kClassWords * 4, "GnClassDev must stay kClassWords words");

// Everything a kernel needs, passed by value (kernel parameter space).
struct GnDev {
    uint32_t N, Npad;        // Npad = N rounded up to 128: one warp of the update kernel owns 128 vertices
    uint32_t D;              // ring slots
    uint32_t words_pad;      // Npad / 32 raster words per step
    uint32_t n_classes;
    uint32_t obs_stride, raster_cap, trace_cap;
    uint32_t seed_lo, seed_hi;
    uint32_t any_drive;      // some class has drive_thr > 0
    float dt, keep_c, ca_jump;
    float obs_gain, obs_offset, obs_sigma, inv_stride;
    // vertex state, SoA, each Npad long
    float *V, *W, *r, *c, *acc, *bias;
    float *p2;               // second PSC state of alpha-function classes (touched only when any_alpha)
    uint32_t any_alpha;
    float *hm, *hh;          // gates m and h of Hodgkin-Huxley vertices (touched only when any_hh); n lives in W
    uint32_t any_hh;
    uint8_t *refr, *cls;
    // delay ring [D][Npad], int32 fixed point 2^-16
    int32_t *ring;
    // CSR by source
    uint32_t *row;           // [Npad + 1]
    uint32_t *tgt;           // [E]
    int32_t *wfx;            // [E]
    uint8_t *dly;            // [E]
    // queue mode: ring slots are taken 2^q_log at a time (a slot GROUP); a spike's events due more than
    // q_window groups ahead are not expanded when it fires but when the group they land in is about to be consumed
    uint32_t queue_mode;     // 0 ring, 1 queue
    uint32_t q_log, q_nb;    // slots per group = 1 << q_log; groups per ring lap = D / 2^q_log
    uint2 *s_edge;           // [E] the CSR rows again, each sorted by delay: {target, w_fx}; when `packed`
                             //     (Npad <= 2^24) the delay also sits in the target word's top byte
    uint8_t *s_dly;          // [E] delay of s_edge[e]
    uint8_t *min_dly;        // [Npad] smallest out-delay of every vertex (255: no out-edge)
    uint32_t packed;
    uint32_t persist;        // ring mode on a network whose update grid is co-resident: gn_persist_kernel steps a whole gn_step call in one cooperative launch
    uint32_t fused;          // ring mode on a small network: the update kernel delivers every event itself (no delivery kernel)
    // resident mode (gn_resident_kernel): every network in one CTA
    uint32_t resident;       // 0 / 1
    uint32_t n_networks;
    uint32_t res_cluster;    // CTAs per network: 1, or a thread-block cluster of up to 16 (1,024 vertices each)
    uint32_t res_threads;    // CTA size = largest network rounded up to 32 (1,024 in cluster mode)
    uint32_t res_smem;       // dynamic shared memory: ring [D][res_threads] + drive words
    const uint32_t *net_off; // [n_networks + 1] first vertex of every network
    uint32_t q_window;       // queue mode, W: the update kernel sends the events due fewer than W groups ahead itself, the
                             //     logging kernel those due exactly W groups ahead; later ones are logged
    uint16_t *q_seg;         // [N][2^q_log][q_nb] segment boundaries of every delay-sorted row (rows of more than 65,535
                             //     edges have no entry: their boundaries are searched for)
    // the spike log: for the spike at position i of step t (slot t mod D) and every group offset j = q_window+1 ..
    // q_nb+1, the index of the first edge of its row due j groups ahead, spk_log[((t mod D) * q_arrays + j-q_window-1)
    // * log_cap + i]; the events due j groups ahead are edges [entry j, entry j+1)
    uint32_t *spk_log;
    uint32_t q_arrays;       // q_nb - q_window + 1 (0 or 1: nothing is ever logged)
    uint32_t log_cap;        // spikes of one step the log holds; later ones are delivered on the spot
    uint32_t *log_n;         // [D] spikes of step (slot) logged or delivered on the spot (may exceed log_cap)
    // plastic mode (gn_config.stdp_alpha != 0; eq. 32-33): weights are state, delivery happens at arrival
    uint32_t plastic;
    float stdp_dta, stdp_beta;      // (float)(dt * alpha), beta
    float *w_f32;                   // [E] current weight of s_edge[e] (the int32 in s_edge[e].y is the initial one)
    uint32_t *perm;                 // [E] caller's edge index of s_edge[e]
    int32_t *ls_hist;               // [D+1][Npad] row t mod (D+1): last spike step of every vertex strictly before t (-1: none)
    uint32_t *pl_list;              // [D][Npad] row t mod D: the vertices that fired at step t (log_n[t mod D] of them)
    uint32_t *csc_off, *csc_edge, *csc_src;   // in-edges by target: [Npad+1] offsets, [E] position in s_edge, [E] source
    float *w_stage;                 // [E] staging of GN_WEIGHTS read-back (caller's edge order)
    unsigned long long *faults;     // [2] GN_FAULTS: deliveries of a weight outside the fixed-point range; targets over gn_create's bound when last evaluated
    unsigned long long *counters;   // steps, spikes, delivered events, kicks
    unsigned long long *grid_sync;  // the persistent step driver's barrier counter (it only grows)
    uint32_t *raster;        // [raster_rows][words_pad]; row t % raster_rows is step t's spike list
    uint32_t raster_rows;    // max(raster_cap, 2): the delivery kernels read the current row even when none is kept
    float *trace;            // [trace_cap][Npad]
    GnClassDev cls_tab[GN_MAX_CLASSES];
};

// Flags written by the create-time validation kernels.
struct GnCheck {
    uint32_t bad_row, bad_target, bad_delay, bad_class, bad_weight, cross_net, overflow;
    uint32_t bad_position;   // a NaN / infinite coordinate reached eq. 25
};

// ---- launchers (gn_kernels.cu).  All asynchronous on `st`; return the launch error. ----
cudaError_t gnk_update(const GnDev &p, uint64_t t, bool has_bias, cudaStream_t st);
cudaError_t gnk_deliver(const GnDev &p, uint64_t t, cudaStream_t st);
// Queue mode.  gnk_log: the spikes of steps t0 .. t0+n_batch-1 (one slot group at most) enter the spike log.
// gnk_fold: for the n_win steps starting at step t_win, the log entries due in absolute slot group g_fold are expanded and
// added into that group's ring rows; beside_previous: it may start while the kernel in front of it in the stream is
// still running (the logging kernel of the same group end, which it does not depend on).
// zero_next: the spike counts of that many steps after the batch are zeroed as well (at most D - n_batch, at most 256)
cudaError_t gnk_log(const GnDev &p, uint64_t t0, uint32_t n_batch, uint32_t zero_next, cudaStream_t st);
cudaError_t gnk_fold(const GnDev &p, uint64_t t_win, uint32_t n_win, uint64_t g_fold, bool beside_previous, cudaStream_t st);
cudaError_t gnk_sort_rows(const GnDev &p, GnCheck *chk, cudaStream_t st);
// plastic mode: in-edge lists (csc_*; csc_off must hold zeros), then per step arrive -> update -> plasticity
cudaError_t gnk_build_csc(const GnDev &p, uint64_t n_edges, uint32_t *cursor, cudaStream_t st);
cudaError_t gnk_arrive(const GnDev &p, uint64_t t, uint64_t t_origin, cudaStream_t st);
cudaError_t gnk_plasticity(const GnDev &p, uint64_t t, uint64_t t_origin, cudaStream_t st);
cudaError_t gnk_weights_out(const GnDev &p, uint64_t n_edges, cudaStream_t st);
// plastic mode: faults[1] = targets whose current sum |w_fx| (+ kick) passes 2^31 - 1; abs_in: N x 8 bytes of scratch
cudaError_t gnk_plastic_headroom(const GnDev &p, uint64_t n_edges, unsigned long long *abs_in, cudaStream_t st);
cudaError_t gnk_observe(const GnDev &p, uint64_t frame, cudaStream_t st);
cudaError_t gnk_resident(const GnDev &p, uint64_t t0, uint32_t n_steps, bool has_bias, bool raster_on, cudaStream_t st);
cudaError_t gnk_resident_cluster_ok(const GnDev &p, bool *ok);
cudaError_t gnk_persist_ok(const GnDev &p, bool *ok);
// sync: a device counter the launch's grid barrier counts on (it only grows); *sync_base: its value before / after the launch
cudaError_t gnk_persist(const GnDev &p, uint64_t t0, uint32_t n_steps, bool has_bias, unsigned long long *sync,
                        unsigned long long *sync_base, cudaStream_t st);
cudaError_t gnk_init_state(const GnDev &p, GnCheck *chk, cudaStream_t st);
cudaError_t gnk_convert_rows(const GnDev &p, const uint64_t *row64, uint64_t n_edges, GnCheck *chk,
                             cudaStream_t st);
cudaError_t gnk_quantise(const GnDev &p, uint64_t n_edges, GnCheck *chk, cudaStream_t st);
cudaError_t gnk_delays_from_positions(const GnDev &p, const float *pos, uint32_t dim, float speed,
                                      GnCheck *chk, cudaStream_t st);
cudaError_t gnk_validate(const GnDev &p, const uint32_t *net_of_vertex_offsets, uint32_t n_networks,
                         unsigned long long *abs_in, GnCheck *chk, cudaStream_t st);
cudaError_t gnk_check_overflow(const GnDev &p, const unsigned long long *abs_in, GnCheck *chk,
                               cudaStream_t st);
cudaError_t gnk_debug_words(uint64_t seed, uint32_t stream_id, uint64_t idx, uint32_t first,
                            uint32_t n, uint32_t *out, cudaStream_t st);
cudaError_t gnk_ceilings(void *scratch, size_t scratch_bytes, uint32_t seg_len, double out[2], cudaStream_t st);
cudaError_t gnk_stream_ceilings(void *scratch, size_t scratch_bytes, double out[2], cudaStream_t st);
// message for gn_last_error(NULL) on this thread; returns `code` (gn_api.cu)
int gn_fail(int code, const char *fmt, ...);
