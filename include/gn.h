/*
 * gn.h -- C ABI of the geometric-network simulation step on one B200 (sm_100a).
 *
 * The operation is the per-timestep transition of Buibas & Silva's framework (arxiv 0908.3934;
 * line numbers below are /root/reference/PAPER.md):
 *
 *   y_j(t + dt) = H_j( y_j(t), Y_j(t), u_j(t), Theta_j )                     :68-71  eq. 5
 *
 * with  y_j = {V, W, r, c} an Izhikevich simple-model vertex with hard reset (:227-229 eq. 24,
 * :303 eq. 28) or a Hodgkin-Huxley vertex {V, m, h, n} (:235, :382), an exponential (:283-286 eq. 26)
 * or alpha-function (:288-312 eq. 27-30, state p) post-synaptic current and a calcium state
 * (:364 H_c); optionally plastic weights w_ij(t) with the STDP transition function (:323-349 eq. 32-33);  Y_j(t) the delayed, weighted spikes of the other vertices,
 * sum_k w_kj spd(V_k(t - tau_kj)) (:311 eq. 30, spd = [V >= V_peak] :316 eq. 31) with
 * tau_kj = |x_k - x_j| / s (:251 eq. 25);  u_j(t) the external control (:77-79 eq. 7); and the
 * observation I_j = n c_j + b + N(0, gamma^2) averaged over camera frames (:370-374).
 * DESIGN.md lists every reading taken where the paper is silent or garbled and the exact fp32
 * operation sequence ("arithmetic contract") the kernels follow.
 *
 * Conventions
 *   - Every function returns GN_OK (0) or a negative GN_E_* code; nothing throws, exits or keeps
 *     global state.  gn_last_error() gives a NUL-terminated message for the last failure on a
 *     handle (or, with NULL, of the last failed gn_create on this thread).
 *   - Memory: the library never allocates device memory.  gn_create carves everything out of a
 *     caller-supplied DEVICE workspace (gn_query_workspace bytes, 256-byte aligned) that must
 *     outlive the handle.  Input arrays of gn_create may be host or device pointers (they are
 *     copied with cudaMemcpyDefault) and may be freed once gn_create returns.
 *   - Streams: all work is enqueued on the cudaStream_t given to gn_create (pass torch's current
 *     stream).  Functions with a host destination synchronise that stream before returning;
 *     device destinations are written asynchronously on it.
 *   - Vertex ids are the caller's.  Step index t counts completed steps from 0.
 *   - There is no CPU fallback: without a CUDA device every call fails with GN_E_CUDA.
 */
#ifndef GN_H_
#define GN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GN_OK 0
#define GN_E_INVALID_ARG (-1)         /* NULL pointer, bad scalar, unsupported size               */
#define GN_E_BAD_GRAPH (-2)           /* row offsets not monotone / target out of range / delay   */
                                      /* 0 or >= ring_slots / edge crossing networks / class id / */
                                      /* NaN or infinite position on an edge when delays == NULL  */
#define GN_E_OVERFLOW_RISK (-3)       /* some target's sum |w_fx| (+ largest kick) >= 2^31        */
#define GN_E_WORKSPACE_TOO_SMALL (-4)
#define GN_E_RANGE_EVICTED (-5)       /* raster / trace range not (or no longer) held             */
#define GN_E_CUDA (-6)                /* a CUDA runtime call failed; see gn_last_error            */

#define GN_MAX_CLASSES 8

typedef struct gn_net gn_net;

/* One vertex class (e.g. 0 = regular-spiking excitatory, 1 = fast-spiking inhibitory).
 * dV/dt = k2 V^2 + k1 V + k0 - W + r + U,  dW/dt = a (b V - W);  V >= v_peak: V <- c_reset,
 * W <- W + d  (eq. 23-24 in its (a,b,c,d) parametrisation, reading #1). */
typedef struct {
    float a, b, c_reset, d;
    float k2, k1, k0, v_peak;
    float tau_syn_ms;       /* exponential PSC time constant 1/a of eq. 26 (:283-286); <= 0 selects  */
                            /* direct injection: the arriving weight jumps V itself                  */
    float refractory_ms;    /* absolute refractory hold after a spike (:259, reading #6)             */
    float drive_rate_hz;    /* Bernoulli(rate*dt) kick per step from the counter generator           */
    float drive_kick;       /* kick weight, injected like an arriving event (reading #12)            */
    float psc_alpha;        /* 0: exponential PSC (eq. 26).  != 0: alpha-function PSC (:288-312 eq. 27,  */
                            /* 29, 30), a = 1/tau_syn_ms: r <- r + dt p, p <- p + dt(-a^2 r - 2a p) + I   */
    /* Vertex model of the class.  0 (GN_MODEL_IZHIKEVICH): the fields above.  1 (GN_MODEL_HODGKIN_HUXLEY): the      */
    /* paper's second benchmarked model (PAPER.md:235 "states {v, m, n, h}", dt ~ 0.03 ms; :382), textbook form:     */
    /*   C dV/dt = -g_na m^3 h (V - e_na) - g_k n^4 (V - e_k) - g_l (V - e_l) + r + U,                               */
    /*   dx/dt = alpha_x(V) (1 - x) - beta_x(V) x  for x = m, h, n,  forward Euler (:184 eq. 19), no reset.          */
    /* Of the fields above it uses v_peak (a spike is V >= v_peak while not in the dead time, eq. 31),               */
    /* refractory_ms (the detection dead time: one action potential is one event), tau_syn_ms, psc_alpha and the     */
    /* drive; a .. k0 are ignored.  The state n is read / written as GN_W, m and h as GN_M and GN_H.                 */
    float model;
    float hh_c;                          /* membrane capacitance, uF/cm^2 (> 0)                                      */
    float hh_g_na, hh_g_k, hh_g_l;       /* maximal conductances, mS/cm^2                                            */
    float hh_e_na, hh_e_k, hh_e_l;       /* reversal potentials, mV                                                  */
    float hh_v_rest;                     /* initial V; the gates start at alpha/(alpha+beta) of this potential        */
    /* The six rate functions, each {A, V_half, k} (k != 0), u = (V - V_half)/k, in 1/ms:                            */
    /*   alpha_m, alpha_n: linoid A k u / (1 - exp(-u)); beta_h: sigmoid A / (1 + exp(-u)); beta_m, alpha_h, beta_n: */
    /*   exponential A exp(-u)                                                                                       */
    float hh_am[3], hh_bm[3], hh_ah[3], hh_bh[3], hh_an[3], hh_bn[3];
} gn_class_params;

#define GN_MODEL_IZHIKEVICH 0
#define GN_MODEL_HODGKIN_HUXLEY 1

typedef struct {
    uint32_t n_vertices;            /* N (total over all networks in batched mode)                   */
    uint32_t dim;                   /* 2 or 3: columns of `positions`                                */
    uint64_t n_edges;               /* E < 2^32                                                      */
    uint32_t n_networks;            /* 1, or B independent networks stepped together (block-diagonal)*/
    uint32_t ring_slots;            /* 2 <= D <= 255; every delay satisfies 1 <= delay <= D-1        */
    float    dt_ms;                 /* time step                                                     */
    float    speed;                 /* conduction speed, position units per ms (delays == NULL)      */
    uint32_t n_classes;             /* 1 .. GN_MAX_CLASSES                                           */
    float    tau_ca_ms, ca_jump;    /* calcium filter c <- c (1 - dt/tau_ca) + ca_jump*fired (:364)  */
    float    obs_gain, obs_offset, obs_sigma;   /* n, b, gamma of I = n c + b + N(0,gamma^2) (:370)  */
    uint32_t obs_stride;            /* steps averaged per camera frame (:374); 0 = observation off   */
    uint32_t raster_capacity_steps; /* device raster window (most recent steps kept); 0 = none kept  */
    uint32_t trace_capacity_frames; /* device trace window (most recent frames kept)                 */
    uint64_t seed;                  /* key of the counter generator (drive stream 5, noise stream 6) */
    /* How eq. 30's sum reaches the ring (the RESULT is identical in every mode: integer adds commute). */
    uint32_t delivery_mode;         /* GN_DELIVER_AUTO (0), _RING, _QUEUE, _RESIDENT, _RING_STEPWISE   */
    uint32_t queue_group;           /* queue mode: ring slots per slot group, power of two in 1..16;  */
                                    /* 0 = default (8)                                                */
    uint64_t queue_capacity;        /* queue mode: spikes of one step the spike log holds; later ones */
                                    /* are expanded on the spot (direct ring adds); 0 = default       */
                                    /* max(1024, N / 16)                                              */
    /* Plasticity (eq. 32-33, readings #22, #23).  stdp_alpha != 0 makes every weight a state   */
    /* of its own: w_ij(t+dt) = w_ij(t) + dt alpha sign(q) exp(-beta |q|), q = s~_i(t - tau_ij) - s~_j(t) whenever the      */
    /* spike of i arrives at j or j fires at t (s~: time since the last spike, 0 for a vertex spiking at the step).  An   */
    /* arriving spike is weighed with the weight AT THE ARRIVAL step (eq. 30), so delivery then happens at arrival time:  */
    /* delivery_mode must be AUTO or RING, and checkpoint writes of RING / STEP / COUNTERS are not supported with it.    */
    /* Overflow: GN_E_OVERFLOW_RISK of gn_create bounds the INITIAL weights only, and eq. 33 has no ceiling.  GN_FAULTS   */
    /* is the guard of a plastic network: [0] counts, at delivery, every weight that no longer fits the fixed point (it is */
    /* delivered saturated); [1] is gn_create's own bound (a target's sum of |w_fx| + kick <= 2^31 - 1, so that no ring    */
    /* slot can wrap) re-evaluated over the current weights whenever GN_FAULTS or GN_WEIGHTS is read -- nothing is added   */
    /* to the step for it, so read one of them as often as the learning rate makes prudent.  A read into HOST memory (of   */
    /* these or of GN_COUNTERS) tells the handle; once a count is non-zero gn_step returns GN_E_OVERFLOW_RISK.             */
    float    stdp_alpha;            /* per ms; 0 = static weights                                     */
    float    stdp_beta;             /* 1/ms, >= 0                                                     */
} gn_config;

/* delivery_mode.
 * RING: every event is one int32 reduction straight into ring[(t+delay) mod D][target], by a delivery kernel
 *   that runs beside the next step's update (best while the ring fits L2).
 * QUEUE: ring slots are taken queue_group at a time (a slot group).  A spike is entered into a spike log -- per group
 *   offset, where in its delay-sorted row the events due that many groups ahead begin -- and its events are expanded
 *   and added ("folded") into the ring group by group, each group just before it is consumed, while the group's rows
 *   sit in L2 (best when the ring is >> L2: no 32-byte DRAM sector read-modify-write per event, and nothing per event
 *   is written or read back).  Logging and folding run once per group of steps; events due in the current or the next
 *   group are sent by the update kernel itself, those due in the group after by the logging kernel.  Needs ring_slots to be a multiple of the group (else a smaller group is taken).
 * RESIDENT: every network (n_networks >= 1) lives in ONE CTA -- or, above 1,024 vertices, one thread-block cluster of
 *   up to 16 CTAs -- for a whole gn_step call: vertex state in registers, the network's delay ring in (distributed)
 *   shared memory, delivery by shared-memory integer atomics, one barrier per step and no per-step kernel launch
 *   (the paper's own workload shape: many networks of <= 1000 vertices).  Needs every network to have <= 16,384
 *   vertices and ring_slots x min(vertices, 1024) x 4 bytes <= 200 KB; otherwise GN_E_INVALID_ARG.
 * AUTO picks RESIDENT whenever it is possible, else QUEUE when the ring exceeds 48 MB and D >= 32, else RING.
 * GN_DRIVER (gn_read_state) tells which step driver a handle ended up with. */
#define GN_DELIVER_AUTO 0
#define GN_DELIVER_RING 1
#define GN_DELIVER_QUEUE 2
#define GN_DELIVER_RESIDENT 3
/* RING with one kernel launch per step even where the whole gn_step call could be one cooperative launch (the persistent
 * step driver, small networks): for measuring and testing the per-step path.  Same results. */
#define GN_DELIVER_RING_STEPWISE 4

/* GN_DRIVER values: which step driver gn_create chose for this network. */
#define GN_DRIVER_RING 0        /* update kernel + delivery kernel per step                                  */
#define GN_DRIVER_FUSED 1       /* one kernel per step, the update delivers                                  */
#define GN_DRIVER_PERSISTENT 2  /* one cooperative launch per gn_step call (gn_persist_kernel)               */
#define GN_DRIVER_QUEUE 3       /* update per step, logging + folding per slot group                         */
#define GN_DRIVER_RESIDENT 4    /* one launch per call, a CTA or cluster per network                         */
#define GN_DRIVER_PLASTIC 5     /* arrival-time delivery, update, eq. 32-33: four launches per step          */

/* `which` of gn_read_state / gn_write_state, with the element type of the caller's buffer.       */
enum {
    GN_V = 0,         /* float  [N]      membrane potential                                          */
    GN_W = 1,         /* float  [N]      recovery variable                                           */
    GN_R = 2,         /* float  [N]      post-synaptic current r                                     */
    GN_CA = 3,        /* float  [N]      calcium c (maintained only when obs_stride > 0)             */
    GN_REFR = 4,      /* uint8  [N]      refractory steps left                                       */
    GN_RING = 5,      /* int32  [D][N]   delay ring, fixed point 2^-16.  After T completed steps     */
                      /*                 slot s holds the arrivals due at steps a = s (mod D),       */
                      /*                 T <= a <= T + D - 2; slot (T-1) mod D is zero               */
    GN_STEP = 6,      /* uint64 [1]      completed steps t                                           */
    GN_COUNTERS = 7,  /* uint64 [4]      { steps, spikes, delivered events, kicks } up to the last completed */
                      /*                 step (reading it first routes any step whose events are pending)  */
    GN_DELAYS = 8,    /* uint8  [E]      per-edge delay in steps (as given, or eq. 25)               */
    GN_WEIGHTS_FX = 9,/* int32  [E]      per-edge weight, rint(w * 2^16)                             */
    GN_BIAS = 10,     /* float  [N]      user control U_j (write only through gn_write_state)        */
    GN_P = 11,        /* float  [N]      second PSC state p of the alpha-function (zero for other classes) */
    GN_ACC = 12,      /* float  [N]      sum of c over the steps of the camera frame in progress (obs_stride > 0) */
    GN_M = 13,        /* float  [N]      sodium activation m of Hodgkin-Huxley vertices (zero for other classes)  */
    GN_H = 14,        /* float  [N]      sodium inactivation h of Hodgkin-Huxley vertices (zero for other classes) */
    GN_WEIGHTS = 15,  /* float  [E]      current weight of every edge, caller's edge order (plastic: evolving; else w_fx 2^-16) */
    GN_DRIVER = 17,   /* uint32 [1]      the step driver in use, a GN_DRIVER_* value (read only)                                */
    GN_FAULTS = 16    /* uint64 [2]      plastic mode's overflow guard (read only; zeros otherwise): { deliveries, since       */
                      /*                 gn_create, of a weight outside the fixed-point range +-32768 (or NaN); targets whose  */
                      /*                 sum of |w_fx| (+ kick) passes 2^31 - 1 for the weights as they are at this read } --  */
                      /*                 see stdp_alpha                                                                         */
};

/* Bytes of device workspace gn_create needs for this configuration.
 * Errors: GN_E_INVALID_ARG (NULL, N = 0, dim not 2/3, D < 2 or > 255, E >= 2^32, n_classes out of
 * range, dt <= 0, obs_stride > 0 with trace_capacity_frames = 0). */
int gn_query_workspace(const gn_config *cfg, size_t *bytes);

/*
 * Build a network on the device.
 *   classes       [n_classes]
 *   positions     [N][dim] float, row-major.  May be NULL when `delays` is given.
 *   row_offsets   [N+1] CSR by SOURCE vertex: out-edges of i are row_offsets[i] .. row_offsets[i+1]-1
 *   targets       [E] target vertex of each edge
 *   weights       [E] fp32; quantised here to int32 fixed point, w_fx = rint(w * 65536) (ties to even)
 *   delays        [E] steps, or NULL => max(1, ceil(|x_i - x_j| / (speed * dt))) in double (eq. 25)
 *   vertex_class  [N] class id < n_classes
 *   bias          [N] constant user control U_j added inside eq. 28's bracket, or NULL (none)
 *   net_offsets   [n_networks + 1] first vertex of each network (batched mode), or NULL when
 *                 n_networks == 1; an edge whose endpoints lie in different networks is rejected
 *   workspace     device memory, >= gn_query_workspace bytes, 256-byte aligned; owned by the caller
 *   cuda_stream   cudaStream_t (NULL = legacy default stream)
 * Initial state (reading #15): V = -70, W = b V, r = c = 0, not refractory, ring empty, t = 0; a Hodgkin-Huxley
 * vertex starts at V = hh_v_rest with m, h, n at their steady states for that potential.
 * Synchronises the stream once (validation results are read back).  On failure *out = NULL.
 * Errors: INVALID_ARG, BAD_GRAPH, OVERFLOW_RISK, WORKSPACE_TOO_SMALL, CUDA.
 */
int gn_create(const gn_config *cfg, const gn_class_params *classes, const float *positions,
              const uint64_t *row_offsets, const uint32_t *targets, const float *weights,
              const uint8_t *delays, const uint8_t *vertex_class, const float *bias,
              const uint32_t *net_offsets, void *workspace, size_t workspace_bytes,
              void *cuda_stream, gn_net **out);

/* Advance n_steps time steps (eq. 5, called in a loop).  Per step one update kernel: ring-slot
 * read-and-clear + drive + vertex update + spike detection + raster word + the events due soonest; then the rest of the
 * step's event delivery -- ring mode: a delivery kernel per step (small networks: inside the update kernel, or the whole
 * call as one cooperative launch); queue mode: one logging and one folding kernel per group of queue_group steps;
 * resident mode: the whole call is one launch per network batch -- and at frame boundaries the observation kernel.
 * Asynchronous: no host synchronisation inside. */
int gn_step(gn_net *net, uint64_t n_steps);

/* Copy state out.  dst_bytes must be at least the size listed at the enum.  dst_is_device != 0:
 * dst is device memory, written asynchronously on the stream.  Errors: INVALID_ARG, CUDA. */
int gn_read_state(gn_net *net, int which, void *dst, size_t dst_bytes, int dst_is_device);

/* Overwrite V, W, R, P, M, H, CA, ACC (float [N]), REFR (uint8 [N]) or BIAS (float [N]; enables the bias term): controlled
 * experiments (PAPER.md:77-79 user control).  Checkpoint / restore: together with RING (int32 [D][N], the layout GN_RING
 * reads) and STEP (uint64 [1], or COUNTERS uint64 [4]) they are the whole state -- y_j and the in-flight delayed signals
 * Y_j: a fresh handle of the same network given all of them continues bit-identically from step t.
 * Writing STEP / COUNTERS sets the step index (generator counter, ring slot, frame phase); raster steps and trace
 * frames before it are not held (GN_E_RANGE_EVICTED).  RING / STEP / COUNTERS writes synchronise the stream.
 * Not covered: a plastic network (stdp_alpha != 0).  Its state also includes the weights (GN_WEIGHTS, read-only), the
 * spikes in flight -- which it keeps as the spike lists of the last ring_slots - 1 steps, not in the ring -- and the
 * last-spike steps of eq. 32; none of these can be written, so RING / STEP / COUNTERS writes are refused there
 * (GN_E_INVALID_ARG) and a plastic run cannot be resumed from a checkpoint. */
int gn_write_state(gn_net *net, int which, const void *src, size_t src_bytes, int src_is_device);

/* Spike raster of steps t0 .. t0+n_steps-1 as bit words: bit (j mod 32) of bits[s][j / 32] is
 * spd(V_j(t0 + s)) (eq. 31); row length ceil(N/32) words.  Errors: RANGE_EVICTED if any step is
 * not yet simulated or older than raster_capacity_steps. */
int gn_read_raster(gn_net *net, uint64_t t0, uint64_t n_steps, uint32_t *bits, size_t dst_bytes,
                   int dst_is_device);

/* Observation trace, frames frame0 .. frame0+n_frames-1, trace[f][j] = I_j of frame f
 * (PAPER.md:370-374); frame f covers steps f*obs_stride .. (f+1)*obs_stride-1.
 * Errors: INVALID_ARG if observation is off, RANGE_EVICTED as for the raster. */
int gn_observe(gn_net *net, uint64_t frame0, uint64_t n_frames, float *trace, size_t dst_bytes,
               int dst_is_device);

/* Test hook: out[i] = 32-bit word of the counter generator for vertex first_vertex + i at index
 * idx on `stream_id` (Philox4x32-10; counter {vertex/4, idx lo, idx hi, stream_id}, key = seed;
 * word vertex mod 4).  `out` is DEVICE memory.  Lets the known-answer vectors reach the device
 * implementation. */
int gn_debug_words(void *cuda_stream, uint64_t seed, uint32_t stream_id, uint64_t idx,
                   uint32_t first_vertex, uint32_t n, uint32_t *out);

/* Benchmark hook: the measured ceilings of event delivery's access pattern on this device, with everything
 * else of the kernels stripped off.  out[0] = scattered int32 reductions per second into a 16 MB region (one per event is
 * the least any atomic delivery does); out[1] = the same with each reduction's 8-byte edge gathered first, in random
 * contiguous segments of `segment_edges` edges from the rest of `scratch` (what folding a slot group does; mean segment
 * = out-degree x queue_group / ring_slots).  `scratch` is DEVICE memory, >= 320 MB (the edge array should dwarf L2), and is
 * overwritten.  Synchronises.  Errors: INVALID_ARG, CUDA. */
int gn_debug_ceilings(void *cuda_stream, void *scratch, size_t scratch_bytes, uint32_t segment_edges, double out[2]);

/* Benchmark hook: the streaming ceilings the update kernel (a1-a3) is rated against, measured on this device with a bare
 * read-modify-write of 128-bit words (every byte read once and written once per pass).  out[0] = bytes/s (read + written)
 * over a 32 MB buffer that stays in L2 between passes -- the update kernel's situation while a network's state fits L2
 * ("limited by memory and bus speeds"; a working set in L2 is rated against L2 bandwidth);
 * out[1] = the same over all of `scratch`, which must be DEVICE memory of >= 1 GB (HBM).  Overwrites scratch; synchronises.
 * Errors: INVALID_ARG, CUDA. */
int gn_debug_stream_ceilings(void *cuda_stream, void *scratch, size_t scratch_bytes, double out[2]);

/* The overflow check of gn_create (GN_E_OVERFLOW_RISK: does any target's sum of |w_fx| over its in-edges, plus the largest
 * drive kick, pass 2^31 - 1 -- the most the int32 ring slot of PAPER.md:311 eq. 30's sum can be asked to hold in one step)
 * as a call of its own that needs NO device memory from the caller beyond the inputs and the 8-byte result.
 *
 * Who it is for: code that cannot allocate on the device when it needs the answer -- a plug-in of a host program whose
 * memory pool owns the whole GPU and forbids driver allocations; a control loop that must not call cudaMalloc / cudaFree
 * because they stall every stream of the device; a process with no memory left once the network's workspace is carved out.
 * Typical use: before gn_create, to learn whether a weight set will be refused without building a workspace for it; and
 * during a plastic run (stdp_alpha != 0), where eq. 33 moves the weights without bound and gn_create's one-time check says
 * nothing about them any more -- read GN_WEIGHTS into a device buffer now and then and pass it here.
 *
 *   targets       [n_edges] DEVICE, target vertex of every edge (any edge order; row offsets are not needed)
 *   weights       [n_edges] DEVICE, fp32, quantised as gn_create does: w_fx = rint(w * 65536), ties to even
 *   largest_kick  the largest |drive_kick| of the classes in use (0 if there is no drive)
 *   out           [2] DEVICE uint32, written asynchronously on cuda_stream (read it after synchronising):
 *                 out[0] = number of targets at risk (0 <=> gn_create would not return GN_E_OVERFLOW_RISK),
 *                 out[1] = number of edges left out because their target is >= n_vertices or their weight is NaN /
 *                          outside the fixed-point range (0 <=> gn_create would not return GN_E_BAD_GRAPH for these reasons)
 *
 * The per-target sums live in a fixed array inside the library image instead of a workspace: GN_STATIC_MAX_VERTICES x 8
 * bytes = 8 MB of every GPU that loads libgn.so, held until the process exits.  Hence:
 *   - n_vertices > GN_STATIC_MAX_VERTICES is refused (GN_E_INVALID_ARG, message names the limit); nothing is truncated;
 *   - no cudaMalloc, cudaFree or other allocating call is made -- two asynchronous memsets and one kernel per call;
 *   - the device that is current when the call is made must be the one cuda_stream, targets, weights and out belong to;
 *   - the first call on each device also looks the array's device address up (cudaGetSymbolAddress); make that first call
 *     before you begin any stream capture;
 *   - every call on a device uses the same array.  It is cleared at the start of each call, so calls one after the other
 *     on one stream are independent, but two calls whose kernels can run at the same time on one GPU (different streams,
 *     different host threads) add into each other's sums and both results are garbage: serialise them yourself.
 * Errors: INVALID_ARG (NULL, n_vertices = 0 or beyond the limit, n_edges >= 2^32 - 1, kick out of range), CUDA. */
#define GN_STATIC_MAX_VERTICES 1048576
int gn_check_headroom_static(void *cuda_stream, uint32_t n_vertices, uint64_t n_edges, const uint32_t *targets,
                             const float *weights, float largest_kick, uint32_t *out);

/* Per-kernel timing for benchmarks.  While enabled, gn_step runs every kernel on the net's stream (no overlap
 * between update and delivery) with a CUDA event wherever the kind of kernel changes, and synchronises every
 * few hundred steps to collect them: a measuring mode, never the mode a throughput number is taken in.  A run
 * of consecutive launches of one kernel (queue mode: the updates of one slot group) is timed as a whole.
 * gn_profile_read: ms[k] = summed device time, launches[k] = launch count of kernel k since the last
 * gn_profile(net, 1): k = 0 update (a1-a3), 1 delivery (a4: ring reductions; queue mode: spike logging, once per group),
 * 2 observation (a5), 3 fold (a4, queue mode: expansion of the log into the ring, once per group).  launches[4] is the total number of kernels this
 * handle has launched since gn_create, profiling or not. */
int gn_profile(gn_net *net, int enable);
int gn_profile_read(gn_net *net, double ms[4], uint64_t launches[5]);

const char *gn_last_error(const gn_net *net);
int gn_destroy(gn_net *net);

#ifdef __cplusplus
}
#endif
#endif /* GN_H_ */
