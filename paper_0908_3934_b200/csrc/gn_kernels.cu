// gn_kernels.cu -- every step of the hot path as hand-written CUDA for sm_100a.
//
//   gn_update_kernel   ring-slot read-and-clear + drive + Izhikevich/PSC/calcium update +
//                      spike detection, raster bits and ballot/popc compaction
//   gn_deliver_kernel  warp-per-active-source CSR expansion, int32 RED into the delay ring  (a4, ring mode)
//   gn_log_kernel, gn_fold_kernel   a4 when the ring is >> L2: spikes are logged, and expanded slot group by slot group
//   gn_resident_kernel / gn_persist_kernel   a1-a5 with no per-step launch (small networks)
//   gn_observe_kernel  frame mean -> gain/offset + Gaussian noise -> trace row              (a5)
//   create-time kernels: row conversion, weight quantisation, eq. 25 delays, validation.
//
// Arithmetic contract: every floating-point operation of the update is an explicit
// round-to-nearest intrinsic in a fixed order, so the result is bit-identical to the fp32-faithful
// CPU oracle.  Delivery and the drive decision are integer; atomics are order-independent.
// Paper line numbers refer to /root/reference/PAPER.md.
#include <cooperative_groups.h>

#include <stdlib.h>

#include <utility>

#include "gn_internal.h"

namespace cg = cooperative_groups;

namespace {

constexpr int kUpdateThreads = 256;          // 8 warps x 128 vertices = 1024 vertices per CTA
constexpr int kVertsPerThread = 4;           // one 128-bit load per SoA array
constexpr int kDeliverThreads = 256;
constexpr uint32_t kStreamDrive = 5, kStreamNoise = 6;

// ---- Philox4x32-10 (Salmon et al., SC'11), from its published description -------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const uint32_t lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// One int32 reduction with no return value (RED.ADD), spelled out.
__device__ __forceinline__ void ring_add(int32_t *cell, const int32_t w)
{
    asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(cell), "r"(w) : "memory");
}

// ---- one vertex, one step: eq. 24 + :303 eq. 28 + :283-286 eq. 26 ------------
// Reads the state at t, writes the state at t+1, returns spd(V(t)) gated by refractoriness.
template <bool BIAS, bool ALPHA>
__device__ __forceinline__ bool vertex_step(const GnClassDev &q, const float dt, const int32_t I_fx,
                                            const float U, float &V, float &W, float &r, uint32_t &refr, float &pp)
{
    const float If = __fmul_rn(__int2float_rn(I_fx), 0x1p-16f);
    const bool fired = (refr == 0u) && (V >= q.v_peak);                  // eq. 31 (>=)
    const float u1 = __fmaf_rn(q.b, V, -W);
    const float u2 = __fmul_rn(q.a, u1);
    const float W_euler = __fmaf_rn(dt, u2, W);                          // eq. 24, W line
    float Vn, Wn;
    if (fired) {                                                         // eq. 24 "otherwise"
        Vn = q.c_reset;
        Wn = __fadd_rn(W, q.d);
        refr = q.R;
    } else if (refr > 0u) {                                              // refractory hold (reading #6)
        Vn = q.c_reset;
        Wn = W_euler;
        refr -= 1u;
    } else {                                                             // eq. 28, V < V_peak
        const float t1 = __fmaf_rn(q.k2, V, q.k1);
        const float t2 = __fmaf_rn(t1, V, q.k0);
        const float t3 = __fsub_rn(t2, W);
        float t4 = q.direct ? t3 : __fadd_rn(t3, r);
        if (BIAS) t4 = __fadd_rn(t4, U);
        Vn = __fmaf_rn(dt, t4, V);
        if (q.direct) Vn = __fadd_rn(Vn, If);
        Wn = W_euler;
    }
    if (ALPHA && q.alpha) {                                              // alpha-function PSC, eq. 27, 29, 30
        const float q1 = __fmul_rn(q.a2, r);
        const float q2 = __fmaf_rn(q.two_a, pp, q1);
        const float p1 = __fmaf_rn(-dt, q2, pp);
        r = __fmaf_rn(dt, pp, r);                                        // H_r = r + dt p
        pp = __fadd_rn(p1, If);                                          // H_p = p + dt(-a^2 r - 2a p) + arrivals
    } else if (!q.direct) {
        r = __fmaf_rn(q.keep_s, r, If);                                  // eq. 26
    }
    V = Vn;
    W = Wn;
    return fired;
}

// ---- Hodgkin-Huxley vertex (textbook equations, forward Euler PAPER.md:184 eq. 19) ----------
// exp of the arithmetic contract: clamp to [-87, 88]; n = rint(x log2 e); r = x - n ln 2 in two steps; degree-7 Taylor
// polynomial of e^r by Horner; scaled by 2^n through the exponent field.  Every step one rounded binary32 operation,
// the same sequence as the oracle's fp32-faithful mode, so Hodgkin-Huxley vertices are bit-exact too.
__device__ __forceinline__ float exp32(float x)
{
    x = fminf(fmaxf(x, -87.0f), 88.0f);
    const float n = rintf(__fmul_rn(x, 0x1.715476p+0f));
    float r = __fmaf_rn(n, -0x1.62e400p-1f, x);
    r = __fmaf_rn(n, -0x1.7f7d1cp-20f, r);
    float p = 0x1.a01a02p-13f;
    p = __fmaf_rn(p, r, 0x1.6c16c2p-10f);
    p = __fmaf_rn(p, r, 0x1.111112p-7f);
    p = __fmaf_rn(p, r, 0x1.555556p-5f);
    p = __fmaf_rn(p, r, 0x1.555556p-3f);
    p = __fmaf_rn(p, r, 0.5f);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    return __fmul_rn(p, __int_as_float((__float2int_rn(n) + 127) << 23));
}

// Rate function F of the six (0 alpha_m, 1 beta_m, 2 alpha_h, 3 beta_h, 4 alpha_n, 5 beta_n) at V.
template <int F>
__device__ __forceinline__ float hh_rate(const GnClassDev &q, const float V)
{
    const float u = __fmul_rn(__fsub_rn(V, q.hh_vh[F]), q.hh_inv_k[F]);
    if (F == 0 || F == 4) {                                   // linoid A k u / (1 - exp(-u)); series near u = 0
        if (fabsf(u) < 0.05f) return __fmul_rn(q.hh_ak[F], __fmaf_rn(u, __fmaf_rn(u, 0x1.555556p-4f, 0.5f), 1.0f));
        return __fmul_rn(q.hh_ak[F], __fdiv_rn(u, __fsub_rn(1.0f, exp32(-u))));
    }
    if (F == 3) return __fdiv_rn(q.hh_ak[F], __fadd_rn(1.0f, exp32(-u)));      // sigmoid
    return __fmul_rn(q.hh_ak[F], exp32(-u));                                    // exponential
}

// One Hodgkin-Huxley vertex, one step: state at t in, state at t+1 out (n lives in W); returns spd(V(t)) outside the
// detection dead time.  No reset: `refr` only keeps one action potential from being detected twice.
template <bool BIAS>
__device__ __forceinline__ bool vertex_step_hh(const GnClassDev &q, const float dt, const int32_t I_fx, const float U,
                                               float &V, float &n, float &r, uint32_t &refr, float &pp, float &m, float &h)
{
    const float If = __fmul_rn(__int2float_rn(I_fx), 0x1p-16f);
    const bool fired = (refr == 0u) && (V >= q.v_peak);                  // eq. 31 (>=)
    if (fired) refr = q.R;
    else if (refr > 0u) refr -= 1u;
    const float am = hh_rate<0>(q, V), bm = hh_rate<1>(q, V), ah = hh_rate<2>(q, V);
    const float bh = hh_rate<3>(q, V), an = hh_rate<4>(q, V), bn = hh_rate<5>(q, V);
    const float m2 = __fmul_rn(m, m), m3 = __fmul_rn(m2, m);
    const float i_na = __fmul_rn(__fmul_rn(__fmul_rn(q.hh_g_na, m3), h), __fsub_rn(V, q.hh_e_na));
    const float n2 = __fmul_rn(n, n), n4 = __fmul_rn(n2, n2);
    const float i_k = __fmul_rn(__fmul_rn(q.hh_g_k, n4), __fsub_rn(V, q.hh_e_k));
    const float i_l = __fmul_rn(q.hh_g_l, __fsub_rn(V, q.hh_e_l));
    float s = __fsub_rn(r, __fadd_rn(__fadd_rn(i_na, i_k), i_l));
    if (BIAS) s = __fadd_rn(s, U);
    float Vn = __fmaf_rn(q.hh_dt_c, s, V);
    if (q.direct) Vn = __fadd_rn(Vn, If);                                // reading #4: the arriving weight jumps V itself
    m = __fmaf_rn(dt, __fmaf_rn(-bm, m, __fmul_rn(am, __fsub_rn(1.0f, m))), m);
    h = __fmaf_rn(dt, __fmaf_rn(-bh, h, __fmul_rn(ah, __fsub_rn(1.0f, h))), h);
    n = __fmaf_rn(dt, __fmaf_rn(-bn, n, __fmul_rn(an, __fsub_rn(1.0f, n))), n);
    if (q.alpha) {
        const float q1 = __fmul_rn(q.a2, r);
        const float q2 = __fmaf_rn(q.two_a, pp, q1);
        const float p1 = __fmaf_rn(-dt, q2, pp);
        r = __fmaf_rn(dt, pp, r);
        pp = __fadd_rn(p1, If);
    } else if (!q.direct) {
        r = __fmaf_rn(q.keep_s, r, If);
    }
    V = Vn;
    return fired;
}

// ---- a1 + a2 + a3 (+ calcium of a5) ---------------------------------------------------------------
// Thread g owns vertices 4g .. 4g+3 (128-bit SoA loads); a warp owns 128 vertices = 4 raster words.
// HH: some class is a Hodgkin-Huxley one (two more fp32 streams, m and h; a vertex takes its class's transition function).
template <bool OBS, bool BIAS, bool FUSED, bool ALPHA, bool HH>
__global__ void __launch_bounds__(kUpdateThreads, HH ? 4 : (FUSED || ALPHA) ? 4 : 8)
gn_update_kernel(const GnDev p, const uint64_t t, const uint32_t slot, const uint32_t raster_row,
                 const uint32_t d_direct)
{
    __shared__ GnClassDev s_cls[GN_MAX_CLASSES];
    // Programmatic dependent launch: the next step's update may start launching now; its prologue (class table,
    // Philox words -- nothing a previous kernel wrote) then overlaps this kernel's tail (see griddepcontrol.wait below).
    asm volatile("griddepcontrol.launch_dependents;");
    for (uint32_t q = threadIdx.x; q < p.n_classes * kClassWords; q += kUpdateThreads)
        reinterpret_cast<uint32_t *>(s_cls)[q] = reinterpret_cast<const uint32_t *>(p.cls_tab)[q];
    __syncthreads();

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t g = blockIdx.x * kUpdateThreads + threadIdx.x;
    const uint32_t j0 = g * kVertsPerThread;
    uint32_t nib = 0u, kicks = 0u;                                        // bit q: vertex j0+q fired / kicked

    // drive words first: they depend on no memory, and their temporaries are dead before the state is loaded
    // (the kernel must fit 32 registers so that all N/4 threads are resident in ONE wave).  One Philox block
    // per 4 vertices, counter {j/4, t lo, t hi, 5}, word j mod 4.
    // The class ids are constant after gn_create, so the Bernoulli kicks (reading #12) are decided here too.
    uchar4 cl4 = make_uchar4(0, 0, 0, 0);
    if (j0 < p.Npad) {
        cl4 = *reinterpret_cast<const uchar4 *>(p.cls + j0);
        if (p.any_drive) {
            uint32_t x[4];
            philox4x32_10(g, (uint32_t)t, (uint32_t)(t >> 32), kStreamDrive, p.seed_lo, p.seed_hi, x);
            const uint32_t cq[4] = {cl4.x, cl4.y, cl4.z, cl4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if ((j0 + q) < p.N && x[q] < s_cls[cq[q]].drive_thr) kicks |= 1u << q;
        }
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");     // everything before this step is complete and visible
    if (j0 < p.Npad) {
        // a1: read this step's ring slot (cleared below, only if something arrived) and the state, all at once
        int4 *slot_ptr = reinterpret_cast<int4 *>(p.ring + (size_t)slot * p.Npad + j0);
        const int4 I4 = *slot_ptr;
        const float4 V4 = *reinterpret_cast<const float4 *>(p.V + j0);
        const float4 W4 = *reinterpret_cast<const float4 *>(p.W + j0);
        const float4 r4 = *reinterpret_cast<const float4 *>(p.r + j0);
        const uchar4 rf4 = *reinterpret_cast<const uchar4 *>(p.refr + j0);
        float4 U4 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (BIAS) U4 = *reinterpret_cast<const float4 *>(p.bias + j0);
        const uint32_t cl[4] = {cl4.x, cl4.y, cl4.z, cl4.w};
        if ((I4.x | I4.y | I4.z | I4.w) != 0) *slot_ptr = make_int4(0, 0, 0, 0);

        int32_t I[4] = {I4.x, I4.y, I4.z, I4.w};
        float V[4] = {V4.x, V4.y, V4.z, V4.w}, W[4] = {W4.x, W4.y, W4.z, W4.w};
        float r[4] = {r4.x, r4.y, r4.z, r4.w}, U[4] = {U4.x, U4.y, U4.z, U4.w};
        float pp[4] = {0.f, 0.f, 0.f, 0.f};
        if (ALPHA) {
            const float4 p4 = *reinterpret_cast<const float4 *>(p.p2 + j0);
            pp[0] = p4.x; pp[1] = p4.y; pp[2] = p4.z; pp[3] = p4.w;
        }
        float gm[4] = {0.f, 0.f, 0.f, 0.f}, gh[4] = {0.f, 0.f, 0.f, 0.f};
        if (HH) {
            const float4 m4 = *reinterpret_cast<const float4 *>(p.hm + j0);
            const float4 h4 = *reinterpret_cast<const float4 *>(p.hh + j0);
            gm[0] = m4.x; gm[1] = m4.y; gm[2] = m4.z; gm[3] = m4.w;
            gh[0] = h4.x; gh[1] = h4.y; gh[2] = h4.z; gh[3] = h4.w;
        }
        uint32_t refr[4] = {rf4.x, rf4.y, rf4.z, rf4.w};

        uint32_t refr_changed = 0u;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const GnClassDev &k = s_cls[cl[q]];
            if ((kicks >> q) & 1u) I[q] += k.kick_fx;
            const uint32_t refr_old = refr[q];
            const bool fired = ((HH && k.hh) ? vertex_step_hh<BIAS>(k, p.dt, I[q], U[q], V[q], W[q], r[q], refr[q], pp[q], gm[q], gh[q])
                                             : vertex_step<BIAS, ALPHA>(k, p.dt, I[q], U[q], V[q], W[q], r[q], refr[q], pp[q])) &&
                               (j0 + q) < p.N;
            refr_changed |= (refr[q] != refr_old);
            if (fired) nib |= 1u << q;
        }
        *reinterpret_cast<float4 *>(p.V + j0) = make_float4(V[0], V[1], V[2], V[3]);
        *reinterpret_cast<float4 *>(p.W + j0) = make_float4(W[0], W[1], W[2], W[3]);
        *reinterpret_cast<float4 *>(p.r + j0) = make_float4(r[0], r[1], r[2], r[3]);
        if (ALPHA) *reinterpret_cast<float4 *>(p.p2 + j0) = make_float4(pp[0], pp[1], pp[2], pp[3]);
        if (HH) {
            *reinterpret_cast<float4 *>(p.hm + j0) = make_float4(gm[0], gm[1], gm[2], gm[3]);
            *reinterpret_cast<float4 *>(p.hh + j0) = make_float4(gh[0], gh[1], gh[2], gh[3]);
        }
        if (refr_changed)
            *reinterpret_cast<uchar4 *>(p.refr + j0) = make_uchar4(refr[0], refr[1], refr[2], refr[3]);
        if (OBS) {                                                            // calcium + frame accumulator
            const float4 c4 = *reinterpret_cast<const float4 *>(p.c + j0);
            const float4 a4 = *reinterpret_cast<const float4 *>(p.acc + j0);
            float c[4] = {c4.x, c4.y, c4.z, c4.w}, acc[4] = {a4.x, a4.y, a4.z, a4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                c[q] = __fmaf_rn(p.keep_c, c[q], ((nib >> q) & 1u) ? p.ca_jump : 0.0f);   // H_c
                acc[q] = __fadd_rn(acc[q], c[q]);
            }
            *reinterpret_cast<float4 *>(p.c + j0) = make_float4(c[0], c[1], c[2], c[3]);
            *reinterpret_cast<float4 *>(p.acc + j0) = make_float4(acc[0], acc[1], acc[2], acc[3]);
        }
    }

    // a3: raster bits.  Lane l holds bits 4*(l%8) .. +3 of word l/8 of this warp's 4 words.  The raster row of
    // step t is also the step's spike list: the delivery kernels compact it (popc prefix) CTA by CTA.
    uint32_t word = nib << (4u * (lane & 7u));
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 1);
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 2);
    word |= __shfl_xor_sync(0xFFFFFFFFu, word, 4);
    if ((lane & 7u) == 0u && j0 < p.Npad)
        p.raster[(size_t)raster_row * p.words_pad + (j0 >> 5)] = word;
    // a4, the urgent part: events due before the delivery kernel of this step is guaranteed to have run are
    // sent by the vertex that fired (rows are sorted by delay: such edges lead the row).  Ring mode: delay 1
    // (d_direct = 2), so that deliver(t) may overlap update(t+1).  Queue mode: every delay that lands in the
    // group being consumed or in the next W - 1 (W = q_window; d_direct = WG - r): the logging kernel at the group's end
    // sends what is due W groups ahead, the fold kernels the rest.
    // FUSED (ring mode, small networks: a step is bound by launch latency, not by work): the whole of a4 happens here,
    // warp-cooperatively -- every fired vertex of the warp in turn, lanes over its row -- and there is no delivery kernel.
    if (FUSED) {
        unsigned long long events = 0ull;
        uint32_t spikes = 0u;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t m = __ballot_sync(0xFFFFFFFFu, (nib >> q) & 1u);
            spikes += __popc(m);
            while (m) {
                const uint32_t src = (j0 - 4u * lane) + 4u * ((uint32_t)__ffs(m) - 1u) + (uint32_t)q;
                m &= m - 1u;
                const uint32_t beg = p.row[src], end = p.row[src + 1];
                for (uint32_t e = beg + lane; e < end; e += 32u) {
                    const uint2 ev = p.s_edge[e];
                    const uint32_t d = p.packed ? ev.x >> 24 : (uint32_t)p.s_dly[e];
                    uint32_t s1 = slot + d;
                    if (s1 >= p.D) s1 -= p.D;
                    atomicAdd(p.ring + (size_t)s1 * p.Npad + (p.packed ? ev.x & 0xFFFFFFu : ev.x), (int32_t)ev.y);
                }
                events += (unsigned long long)(end - beg);
            }
        }
        if (lane == 0 && spikes) {
            atomicAdd(&p.counters[1], (unsigned long long)spikes);
            atomicAdd(&p.counters[2], events);
        }
    } else if (nib) {
        const uchar4 md4 = *reinterpret_cast<const uchar4 *>(p.min_dly + j0);   // smallest out-delay of each vertex
        const uint32_t md[4] = {md4.x, md4.y, md4.z, md4.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (!((nib >> q) & 1u) || md[q] >= d_direct) continue;          // most vertices have no such edge
            const uint32_t end = p.row[j0 + q + 1];
            for (uint32_t e = p.row[j0 + q]; e < end; ++e) {
                const uint2 ev = p.s_edge[e];
                const uint32_t d = p.packed ? ev.x >> 24 : (uint32_t)p.s_dly[e];
                if (d >= d_direct) break;
                uint32_t s1 = slot + d;
                if (s1 >= p.D) s1 -= p.D;
                atomicAdd(p.ring + (size_t)s1 * p.Npad + (p.packed ? ev.x & 0xFFFFFFu : ev.x), (int32_t)ev.y);
            }
        }
    }
    if (__any_sync(0xFFFFFFFFu, kicks != 0u)) {                           // rare: one atomic per warp with a kick
        const uint32_t warp_kicks = __reduce_add_sync(0xFFFFFFFFu, __popc(kicks));
        if (lane == 0) atomicAdd(&p.counters[3], (unsigned long long)warp_kicks);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) p.counters[0] = t + 1ull;
}

// ---- a3 (compaction) shared by the delivery kernels ------------------------------------------------------
// The step's raster row is its spike list.  A delivery CTA owns kChunkWords-or-fewer consecutive raster
// words (chosen on the host so the grid covers the row) and compacts the set bits into a shared-memory
// source list with a popc prefix scan: no global list, no global cursor.  Returns the number of sources.
constexpr uint32_t kMaxChunkWords = 128;                 // 4096 vertices per CTA at most

// CTA-wide exclusive prefix sum of one count per thread; returns the CTA total (CTA-uniform), `off` = this thread's offset.
template <int THREADS>
__device__ __forceinline__ uint32_t gather_scan(const uint32_t pc, uint32_t *s_wsum, uint32_t &off)
{
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t incl = pc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += v;
    }
    __syncthreads();                                       // s_wsum may still be read from the previous scan
    if (lane == 31u) s_wsum[warp] = incl;
    __syncthreads();
    uint32_t total = 0u;
    off = incl - pc;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) {
        const uint32_t c = s_wsum[w];
        if ((uint32_t)w < warp) off += c;
        total += c;
    }
    return total;                                          // CTA-uniform
}

// Append this thread's fired vertices to the list at base + off (and tag them with `step` when asked).
__device__ __forceinline__ void gather_write(uint32_t word, const uint32_t w0, uint32_t pos, uint32_t *s_list,
                                             uint8_t *s_step, const uint32_t step)
{
    const uint32_t j_base = (w0 + threadIdx.x) << 5;
    while (word) {
        const uint32_t bit = (uint32_t)__ffs(word) - 1u;
        s_list[pos] = j_base + bit;
        if (s_step) s_step[pos] = (uint8_t)step;
        ++pos;
        word &= word - 1u;
    }
}

template <int THREADS>
__device__ __forceinline__ uint32_t gather_sources(const uint32_t *__restrict__ raster_row, const uint32_t w0,
                                                   const uint32_t n_words, uint32_t *s_list, uint32_t *s_wsum)
{
    const uint32_t word = (threadIdx.x < n_words) ? raster_row[w0 + threadIdx.x] : 0u;
    uint32_t off;
    const uint32_t total = gather_scan<THREADS>(__popc(word), s_wsum, off);
    gather_write(word, w0, off, s_list, nullptr, 0u);
    __syncthreads();
    return total;
}

// ---- a4: event delivery, ring mode ---------------------------------------------------------------------
// One warp per fired source; lanes stride over the source's CSR row (coalesced target / weight /
// delay reads); each edge is one int32 reduction (RED.ADD, no return) into ring[(t+delay) mod D][tgt].
// PAPER.md:311 eq. 30 / :297.
__global__ void __launch_bounds__(kDeliverThreads)
gn_deliver_kernel(const GnDev p, const uint32_t slot_t, const uint32_t raster_row, const uint32_t chunk_words)
{
    __shared__ uint32_t s_list[kMaxChunkWords * 32];
    __shared__ uint32_t s_wsum[kDeliverThreads / 32];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t w0 = blockIdx.x * chunk_words;
    const uint32_t n_words = min(chunk_words, p.words_pad - w0);
    const uint32_t n = gather_sources<kDeliverThreads>(p.raster + (size_t)raster_row * p.words_pad, w0, n_words,
                                                       s_list, s_wsum);
    if (n == 0u) return;
    const uint32_t *__restrict__ row = p.row;
    const uint2 *__restrict__ edge = p.s_edge;
    const uint8_t *__restrict__ dly = p.s_dly;
    unsigned long long events = 0ull;
    for (uint32_t idx = warp; idx < n; idx += kDeliverThreads / 32) {
        const uint32_t src = s_list[idx];
        const uint32_t beg = row[src], end = row[src + 1];
        for (uint32_t e = beg + lane; e < end; e += 32u) {
            const uint2 ev = edge[e];
            const uint32_t d = dly[e];
            uint32_t s = slot_t + d;
            if (s >= p.D) s -= p.D;
            if (d != 1u)                                                   // delay 1 was sent by the update kernel
                atomicAdd(p.ring + (size_t)s * p.Npad + (p.packed ? ev.x & 0xFFFFFFu : ev.x), (int32_t)ev.y);
        }
        events += (unsigned long long)(end - beg);
    }
    if (lane == 0 && events) atomicAdd(&p.counters[2], events);
    if (threadIdx.x == 0) atomicAdd(&p.counters[1], (unsigned long long)n);
}

// ---- a4, queue mode: deferred expansion ------------------------------------------------------------------
// When the ring is far larger than L2 a direct reduction costs a 32-byte DRAM sector fetch and a write-back per
// event.  Queue mode defers the EXPANSION of a spike instead: ring slots are taken G = 2^q_log at a time (a slot
// group; nb = D / G groups per lap), and the events of a spike are added to the ring group by group, each group
// just before it is consumed, when its G rows sit in L2.  Integer adds commute, so the ring word a vertex consumes
// holds exactly what direct delivery would have put there (eq. 30).
//
// Rows are sorted by delay at create time, so the events of a spike at step t (r = t mod G) that land j groups
// ahead -- delays [jG - r, (j+1)G - r) -- are one contiguous SEGMENT of its row, and the segment boundaries depend
// only on r: q_seg[(src * G + r) * nb + j-1] = #edges of src with delay < jG - r (create time).
//     j = 0 .. W-1          (W = q_window) sent by the update kernel itself when the vertex fires
//     j = W                 sent by the logging kernel of the spike's group (it runs a whole group before group h+W is read)
//     j = W+1 .. nb         logged: the spike's entry in log array j-W-1 is the (absolute) index of the segment's first
//                           edge, array j-W its end; j = nb is the wrapped tail (r + delay >= D: the group's own rows,
//                           consumed on the next lap)
// One launch per slot group h, after the group's last update, beside the updates of group h+1:
//   LOGGING CTAs  compact the raster rows of the group's steps (a3: popc prefix, no global list), reserve log
//                 positions with one atomic per step and CTA, send the spike's events due W groups ahead and write
//                 nb-W+1 words per spike (a spike beyond the log's capacity is expanded on the spot, into the ring);
//   FOLDING CTAs  take group g = h+W, due to be consumed one group later: for every step of groups g-nb .. g-W-1
//                 (all logged by earlier launches) and every spike of it, the segment due in g -- two coalesced log
//                 reads -- is expanded: one 8-byte edge load and one int32 RED per event into rows that stay in L2.
// No per-event record is written or read back, no per-event reservation: per event DRAM moves the 8-byte edge once
// (in segments of ~G/D of a row) plus ~8/segment-length bytes of log.
constexpr int kRouteThreads = 256;
constexpr int kRouteWarps = kRouteThreads / 32;
constexpr uint32_t kMaxWindow = 256;                    // steps one fold looks back over: (nb - W) G < D <= 255
constexpr int kFoldUnroll = 4;                          // rounds of edge loads in flight per folding warp
constexpr int kFoldCtasPerSm = 4;                       // folding CTAs per SM (persistent)

// #edges of the delay-sorted row [beg, beg+deg) with delay < thr.  Rows of up to 65,535 edges read it from the table
// (entry k of the row's (src, r) line is the count for thr = (k+1)G - r); longer rows search for it.
template <bool PACKED>
__device__ __forceinline__ uint32_t seg_bound(const GnDev &p, const uint16_t *__restrict__ line, const uint32_t k,
                                              const uint32_t thr, const uint32_t beg, const uint32_t deg)
{
    if (deg <= 0xFFFFu) return (uint32_t)__ldg(line + k);
    uint32_t lo = 0u, hi = deg;
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        const uint32_t d = PACKED ? __ldg(&p.s_edge[beg + mid].x) >> 24 : (uint32_t)__ldg(p.s_dly + beg + mid);
        if (d < thr) lo = mid + 1u; else hi = mid;
    }
    return lo;
}

// One spike per lane (`valid`): the row bounds of the fired vertex and two words of its line of the segment table are
// requested: where the events due exactly q_window groups ahead begin (lo_v) and end (first_v = where the logged ones
// begin).  Nothing here depends on the spike's log position.
__device__ __forceinline__ void log_load(const GnDev &p, const uint32_t r, const uint32_t src, const bool valid, uint32_t &beg,
                                         uint32_t &deg, uint32_t &lo_v, uint32_t &first_v)
{
    beg = deg = lo_v = first_v = 0u;
    if (valid) {
        beg = p.row[src];
        deg = p.row[src + 1] - beg;
        lo_v = first_v = deg;
        if (deg <= 0xFFFFu) {
            const uint16_t *line = p.q_seg + (((size_t)src << p.q_log) + r) * p.q_nb;
            if (p.q_window - 1u < p.q_nb) lo_v = (uint32_t)__ldg(line + p.q_window - 1u);
            if (p.q_window < p.q_nb) first_v = (uint32_t)__ldg(line + p.q_window);
        }
    }
}

// ... then (whole warps only), with r = sl mod G and W = q_window:
//   the events due exactly W groups ahead -- edges [lo_v, first_v) of the row, about one per spike -- are sent here, straight
//   into the ring (the update kernel sends only what is due sooner: this launch runs a whole group before their slots are read);
//   the spike is entered into the log of step slot `sl` at position `pos`: its nb-W+1 entries are stored by its lane -- lanes
//   hold consecutive positions, so every array receives one coalesced run per warp.
// The rest is rare and done by the whole warp, spike after spike: rows too long for the table (their boundaries are searched
// for, one per lane), and spikes beyond the log's capacity (expanded now, straight into the ring).
template <bool PACKED>
__device__ __forceinline__ void log_store(const GnDev &p, const uint32_t sl, const uint32_t r, const uint32_t src, const bool valid,
                                          const uint32_t beg, const uint32_t deg, const uint32_t lo_v, const uint32_t first_v,
                                          const uint32_t pos)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t G = 1u << p.q_log, nb = p.q_nb, W = p.q_window, A = p.q_arrays;
    auto send = [&](const uint32_t e) {
        const uint2 ev = __ldg(p.s_edge + e);
        const uint32_t d = PACKED ? ev.x >> 24 : (uint32_t)__ldg(p.s_dly + e);
        uint32_t s1 = sl + d;
        if (s1 >= p.D) s1 -= p.D;
        atomicAdd(p.ring + (size_t)s1 * p.Npad + (PACKED ? ev.x & 0xFFFFFFu : ev.x), (int32_t)ev.y);
    };
    const bool in_table = valid && deg <= 0xFFFFu, logged = valid && pos < p.log_cap;
    if (in_table)
        for (uint32_t x = lo_v; x < first_v; ++x) send(beg + x);
    const uint16_t *line = p.q_seg + ((size_t)src * G + r) * nb;
    if (A >= 2u && in_table && logged) {
        uint32_t *dst = p.spk_log + ((size_t)sl * A) * p.log_cap + pos;
        dst[0] = beg + first_v;
#pragma unroll 6
        for (uint32_t a = 1u; a + 1u < A; ++a) dst[(size_t)a * p.log_cap] = beg + (uint32_t)__ldg(line + W + a);
        dst[(size_t)(A - 1u) * p.log_cap] = beg + deg;
    }
    for (uint32_t m = __ballot_sync(0xFFFFFFFFu, valid && (!in_table || (A >= 2u && !logged))); m; m &= m - 1u) {
        const int sq = __ffs(m) - 1;
        const uint32_t b2 = __shfl_sync(0xFFFFFFFFu, beg, sq), d2 = __shfl_sync(0xFFFFFFFFu, deg, sq);
        const uint32_t src2 = __shfl_sync(0xFFFFFFFFu, src, sq), pos2 = __shfl_sync(0xFFFFFFFFu, pos, sq);
        uint32_t x_w = __shfl_sync(0xFFFFFFFFu, first_v, sq);       // where the logged events begin
        const uint16_t *line2 = p.q_seg + ((size_t)src2 * G + r) * nb;
        auto bound = [&](const uint32_t k) { return k < nb ? seg_bound<PACKED>(p, line2, k, (k + 1u) * G - r, b2, d2) : d2; };
        if (d2 > 0xFFFFu) {                               // a long row: its events due W groups ahead, by the warp
            x_w = bound(W);
            for (uint32_t x = bound(W - 1u) + lane; x < x_w; x += 32u) send(b2 + x);
        }
        if (A < 2u) continue;                             // nothing is ever logged
        if (pos2 < p.log_cap) {                           // (a long row: an in-table row with a position was logged above)
            uint32_t *dst2 = p.spk_log + ((size_t)sl * A) * p.log_cap + pos2;
            for (uint32_t a = lane; a < A; a += 32u) dst2[(size_t)a * p.log_cap] = b2 + bound(W + a);
        } else {
            for (uint32_t x = x_w + lane; x < d2; x += 32u) send(b2 + x);
        }
    }
}

// Logging CTA: the spikes of ONE step (the i-th of the launch: slot0 = t0 mod D, raster row (row0 + i) mod raster_rows)
// among kLogWarps x 32 consecutive raster words.  a3's compaction happens here: popc prefix over the lanes' words and
// over the CTA's warps, ONE reservation (atomic) per CTA for its spikes' log positions -- every warp a stretch of it --
// the fired vertices listed in shared memory; then one lane per spike (log_load, log_store).  The counters take one
// atomic per CTA as well: thousands of same-address atomics serialise in the L2.
constexpr int kLogWarps = 8;

template <bool PACKED>
__device__ __forceinline__ void log_spikes(const GnDev &p, const uint32_t slot0, const uint32_t row0, const uint32_t n_batch)
{
    __shared__ uint16_t s_src[kLogWarps][1024];          // fired vertices of the warp's 1,024, as offsets (16 KB: 8 CTAs per SM)
    __shared__ uint32_t s_tot[kLogWarps], s_base;
    __shared__ unsigned long long s_events;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t ctas_per_step = (p.words_pad + kLogWarps * 32u - 1u) / (kLogWarps * 32u);
    const uint32_t i = blockIdx.x / ctas_per_step;       // (the grid is n_batch x ctas_per_step CTAs)
    const uint32_t w = ((blockIdx.x - i * ctas_per_step) * kLogWarps + warp) * 32u + lane;
    uint32_t sl = slot0 + i, rr = row0 + i;
    if (sl >= p.D) sl -= p.D;
    if (rr >= p.raster_rows) rr -= p.raster_rows;
    uint32_t word = w < p.words_pad ? p.raster[(size_t)rr * p.words_pad + w] : 0u;
    const uint32_t pc = __popc(word);
    uint32_t incl = pc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += v;
    }
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    if (lane == 0u) s_tot[warp] = total;
    if (threadIdx.x == 0) s_events = 0ull;
    const uint32_t v_warp = (w - lane) << 5;              // first vertex of the warp's 32 words
    for (uint32_t k = incl - pc; word; ++k, word &= word - 1u) s_src[warp][k] = (uint16_t)((lane << 5) + (uint32_t)__ffs(word) - 1u);
    __syncthreads();
    uint32_t before = 0u, cta_total = 0u;                 // spikes of the warps in front of this one, of the whole CTA
#pragma unroll
    for (int k = 0; k < kLogWarps; ++k) {
        const uint32_t c = s_tot[k];
        if ((uint32_t)k < warp) before += c;
        cta_total += c;
    }
    if (cta_total == 0u) return;                          // CTA-uniform
    if (threadIdx.x == 0) s_base = atomicAdd(&p.log_n[sl], cta_total);   // its result is needed only when the first entries are stored
    const uint32_t r = sl & ((1u << p.q_log) - 1u);       // D is a multiple of G: slot mod G = t mod G
    // the first 32 spikes of every warp: their loads go out before anybody waits for the reservation
    const bool valid0 = lane < total;
    const uint32_t src0 = valid0 ? v_warp + s_src[warp][lane] : 0u;
    uint32_t beg, deg, lo_v, first_v;
    log_load(p, r, src0, valid0, beg, deg, lo_v, first_v);
    unsigned long long events = (unsigned long long)deg;
    __syncthreads();
    const uint32_t base = s_base + before;
    log_store<PACKED>(p, sl, r, src0, valid0, beg, deg, lo_v, first_v, base + lane);
    for (uint32_t q0 = 32u; q0 < total; q0 += 32u) {      // (a burst: more than 32 spikes among the warp's 1,024 vertices)
        const uint32_t q = q0 + lane;
        const bool valid = q < total;
        const uint32_t src = valid ? v_warp + s_src[warp][q] : 0u;
        log_load(p, r, src, valid, beg, deg, lo_v, first_v);
        events += (unsigned long long)deg;
        log_store<PACKED>(p, sl, r, src, valid, beg, deg, lo_v, first_v, base + q);
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) events += __shfl_xor_sync(0xFFFFFFFFu, events, o);
    if (lane == 0u && events) atomicAdd(&s_events, events);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_events) atomicAdd(&p.counters[2], s_events);
        atomicAdd(&p.counters[1], (unsigned long long)cta_total);
    }
}

// Folding warp fw of n_fw: the log entries of the n_win steps starting at slot win_slot0 (step t_win, r_win = t_win
// mod G) that are due j_first - (groups since t_win's) groups ahead, i.e. in the group being folded.
// A warp takes 32 consecutive (spike, segment) pairs at a time -- two coalesced log reads per lane -- and lays their
// edges out back to back (the chunk's EXPANSION, T slots): slot x belongs to the pair whose segment ends first at or
// after x.  The ends are marked in a shared-memory bit mask, so the owner of a slot is a popc away: rank = ends before
// the slot's 32-slot word (s_rank) + ends before it inside the word; the pair's {edge index - slot, step slot} sits at
// that rank in s_pair (empty segments are not listed).  Every lane of every reduction carries one event; kFoldUnroll
// 32-slot words of edge loads are in flight before their reductions are issued.  Segments of more than kFoldLong edges
// (hubs) are not laid out: the whole warp walks them one after another.
constexpr uint32_t kFoldLong = 64;

// s_pref[i] = spikes logged in the window's steps before step i (i < n_win), P their total; s_pair (32 entries), s_ends
// and s_rank (kFoldLong words each) are this warp's tables.
template <bool PACKED>
__device__ __forceinline__ void fold_chunks(const GnDev &p, const uint32_t *s_pref, const uint32_t P, const uint32_t win_slot0,
                                            const uint32_t n_win, const uint32_t r_win, const uint32_t j_first, const uint32_t fw,
                                            const uint32_t n_fw, uint2 *s_pair, uint32_t *s_ends, uint32_t *s_rank)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t A = p.q_arrays, W = p.q_window;
    const uint2 *__restrict__ edge = p.s_edge;
    const uint8_t *__restrict__ dly = p.s_dly;
    const uint32_t n_chunks = (P + 31u) / 32u;

    // this lane's (spike, segment) pair of chunk c: first edge, edge count, slot of the spike's step
    auto load_pair = [&](const uint32_t c, uint32_t &b, uint32_t &cnt, uint32_t &tsl) {
        b = cnt = tsl = 0u;
        if (c >= n_chunks) return;
        uint32_t lo = 0u, hi = n_win;                     // the step of the chunk's first pair (warp-uniform search) ...
        while (hi - lo > 1u) {
            const uint32_t mid = (lo + hi) >> 1;
            if (s_pref[mid] <= c * 32u) lo = mid; else hi = mid;
        }
        const uint32_t pidx = c * 32u + lane;
        if (pidx >= P) return;
        while (lo + 1u < n_win && s_pref[lo + 1u] <= pidx) ++lo;   // ... and of this lane's (a chunk rarely straddles steps)
        const uint32_t a = j_first - ((r_win + lo) >> p.q_log) - W - 1u;
        tsl = win_slot0 + lo;
        if (tsl >= p.D) tsl -= p.D;
        const uint32_t *L = p.spk_log + ((size_t)tsl * A + a) * p.log_cap + (pidx - s_pref[lo]);
        b = __ldcs(L);
        cnt = __ldcs(L + p.log_cap) - b;
    };
    // one edge: the reduction into ring[(step + delay) mod D][target]
    auto deliver = [&](const uint2 ev, const uint32_t d, const uint32_t tsl) {
        uint32_t s1 = tsl + d;
        if (s1 >= p.D) s1 -= p.D;
        atomicAdd(p.ring + (size_t)s1 * p.Npad + (PACKED ? ev.x & 0xFFFFFFu : ev.x), (int32_t)ev.y);
    };
    uint32_t b, cnt, tsl;
    load_pair(fw, b, cnt, tsl);
    for (uint32_t c = fw; c < n_chunks; c += n_fw) {
        uint32_t nx_b, nx_cnt, nx_tsl;
        load_pair(c + n_fw, nx_b, nx_cnt, nx_tsl);        // the next chunk's entries are on their way during this one
        const uint32_t small = cnt <= kFoldLong ? cnt : 0u;
        uint32_t incl = small;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += v;
        }
        const uint32_t T = __shfl_sync(0xFFFFFFFFu, incl, 31);
        if (T) {
            const uint32_t n_words = (T + 31u) >> 5;      // <= kFoldLong
            const uint32_t listed = __ballot_sync(0xFFFFFFFFu, small != 0u);
            __syncwarp();                                 // the previous chunk's tables are no longer read
            s_ends[lane] = 0u;
            s_ends[lane + 32u] = 0u;
            __syncwarp();
            if (small) {
                s_pair[__popc(listed & ((1u << lane) - 1u))] = make_uint2(b - (incl - small), tsl);
                atomicOr(&s_ends[(incl - 1u) >> 5], 1u << ((incl - 1u) & 31u));
            }
            __syncwarp();
            uint32_t before = 0u;                         // ends before each word: prefix popc over the mask words
#pragma unroll
            for (int half = 0; half < (int)kFoldLong / 32; ++half) {
                const uint32_t pc = __popc(s_ends[lane + 32u * half]);
                uint32_t inc2 = pc;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc2, o);
                    if (lane >= (uint32_t)o) inc2 += v;
                }
                s_rank[lane + 32u * half] = before + inc2 - pc;
                before += __shfl_sync(0xFFFFFFFFu, inc2, 31);
            }
            __syncwarp();
            for (uint32_t w0 = 0u; w0 < n_words; w0 += kFoldUnroll) {
                uint2 ev[kFoldUnroll];
                uint32_t d[kFoldUnroll], sl[kFoldUnroll];
#pragma unroll
                for (int u = 0; u < kFoldUnroll; ++u) {   // all loads of kFoldUnroll words first
                    const uint32_t w = w0 + (uint32_t)u, x = (w << 5) + lane;
                    ev[u] = make_uint2(0u, 0u);
                    d[u] = sl[u] = 0u;
                    if (x < T) {
                        const uint32_t rk = s_rank[w] + __popc(s_ends[w] & ((1u << lane) - 1u));
                        const uint2 pr = s_pair[rk];
                        const uint32_t e = pr.x + x;      // 32-bit on purpose: pr.x = first edge - first slot may have wrapped
                        sl[u] = pr.y;
                        ev[u] = __ldcs(edge + e);
                        d[u] = PACKED ? ev[u].x >> 24 : (uint32_t)__ldg(dly + e);
                    }
                }
#pragma unroll
                for (int u = 0; u < kFoldUnroll; ++u)
                    if (d[u]) deliver(ev[u], d[u], sl[u]);    // a delay is never 0
            }
        }
        for (uint32_t m = __ballot_sync(0xFFFFFFFFu, cnt > kFoldLong); m; m &= m - 1u) {   // long segments, one after another
            const int src = __ffs(m) - 1;
            const uint32_t pb = __shfl_sync(0xFFFFFFFFu, b, src), pn = __shfl_sync(0xFFFFFFFFu, cnt, src);
            const uint32_t ps = __shfl_sync(0xFFFFFFFFu, tsl, src);
            for (uint32_t x = lane; x < pn; x += 32u) {
                const uint2 e2 = __ldcs(edge + pb + x);
                deliver(e2, PACKED ? e2.x >> 24 : (uint32_t)__ldg(dly + pb + x), ps);
            }
        }
        b = nx_b; cnt = nx_cnt; tsl = nx_tsl;
    }
}

// The counts of the window's steps -> s_pref (CTA-wide, kRouteThreads threads), then the chunks.
template <bool PACKED>
__device__ __forceinline__ void fold_group(const GnDev &p, const uint32_t win_slot0, const uint32_t n_win, const uint32_t r_win,
                                           const uint32_t j_first, const uint32_t fw, const uint32_t n_fw)
{
    __shared__ uint32_t s_pref[kMaxWindow];
    __shared__ uint32_t s_wsum2[kRouteWarps];
    __shared__ uint2 s_pair[kRouteWarps][32];
    __shared__ uint32_t s_ends[kRouteWarps][kFoldLong], s_rank[kRouteWarps][kFoldLong];
    const uint32_t warp = threadIdx.x >> 5;
    uint32_t cnt_step = 0u;
    if (threadIdx.x < n_win) {
        uint32_t sl = win_slot0 + threadIdx.x;
        if (sl >= p.D) sl -= p.D;
        cnt_step = min(p.log_n[sl], p.log_cap);
    }
    uint32_t off;
    const uint32_t P = gather_scan<kRouteThreads>(cnt_step, s_wsum2, off);
    s_pref[threadIdx.x] = off;
    __syncthreads();
    if (P == 0u) return;
    fold_chunks<PACKED>(p, s_pref, P, win_slot0, n_win, r_win, j_first, fw, n_fw, s_pair[warp], s_ends[warp], s_rank[warp]);
}

// Queue-mode delivery, first half: the spikes of steps t0 .. t0+n_batch-1 (all inside one slot group) enter the log.
// Launched just before gn_fold_kernel, which does not depend on it (it reads older log entries only): the trigger lets
// the two run side by side.
template <bool PACKED>
__global__ void __launch_bounds__(kLogWarps * 32, 8)     // 984 CTAs at config 4: one wave, so that the fold behind it starts at once
gn_log_kernel(const GnDev p, const uint32_t slot0, const uint32_t row0, const uint32_t n_batch, const uint32_t zero_next)
{
    asm volatile("griddepcontrol.launch_dependents;");
    // the spike counts of the zero_next steps after this batch are zeroed for the next launch (their slots hold the counts of
    // D steps earlier, which no fold still to come reads: the launcher checks that)
    if (blockIdx.x == 0 && threadIdx.x < zero_next) {
        uint32_t sl = slot0 + n_batch + threadIdx.x;
        while (sl >= p.D) sl -= p.D;
        p.log_n[sl] = 0u;
    }
    log_spikes<PACKED>(p, slot0, row0, n_batch);
}

// Queue-mode delivery, second half: one slot group folded out of the log (persistent CTAs, grid-stride over the log).
template <bool PACKED>
__global__ void __launch_bounds__(kRouteThreads, kFoldCtasPerSm)
gn_fold_kernel(const GnDev p, const uint32_t win_slot0, const uint32_t n_win, const uint32_t r_win, const uint32_t j_first)
{
    fold_group<PACKED>(p, win_slot0, n_win, r_win, j_first, blockIdx.x * kRouteWarps + (threadIdx.x >> 5), gridDim.x * kRouteWarps);
}

// ---- create time, queue mode: copy every CSR row sorted by delay (counting sort, one warp per row) --------
__global__ void __launch_bounds__(256)
gn_sort_rows_kernel(const GnDev p, GnCheck *chk)
{
    __shared__ uint32_t s_hist[8][256];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t *h = s_hist[warp];
    const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < p.N; i += n_warps) {
        const uint32_t beg = p.row[i], end = p.row[i + 1];
#pragma unroll
        for (int k = 0; k < 8; ++k) h[lane * 8 + k] = 0u;
        __syncwarp();
        uint32_t dmin = 255u;
        for (uint32_t e = beg + lane; e < end; e += 32u) {
            const uint32_t d = p.dly[e];
            atomicAdd(&h[d], 1u);
            dmin = min(dmin, d);
        }
        dmin = __reduce_min_sync(0xFFFFFFFFu, dmin);
        if (lane == 0) p.min_dly[i] = (uint8_t)dmin;
        __syncwarp();
        uint32_t c[8], sum = 0u;
#pragma unroll
        for (int k = 0; k < 8; ++k) { c[k] = h[lane * 8 + k]; sum += c[k]; }
        uint32_t incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += v;
        }
        uint32_t run = incl - sum;
#pragma unroll
        for (int k = 0; k < 8; ++k) { h[lane * 8 + k] = run; run += c[k]; }
        __syncwarp();
        // h[d] = #edges with delay < d.  Segment table (see log_spikes): entry (r, k) = h[(k+1)G - r].
        if (p.q_seg) {
            const uint32_t G = 1u << p.q_log, nb = p.q_nb, deg = end - beg;
            // (a row of more than 65,535 edges cannot be described in 16 bits: its entries are never read, see seg_bound)
            uint16_t *seg = p.q_seg + (size_t)i * G * nb;
            for (uint32_t x = lane; x < G * nb; x += 32u) {
                const uint32_t r = x / nb, k = x - r * nb;
                const uint32_t dd = (k + 1u) * G - r;
                seg[x] = (uint16_t)(dd >= p.D ? deg : h[dd]);
            }
        }
        __syncwarp();
        for (uint32_t e = beg + lane; e < end; e += 32u) {
            const uint32_t d = p.dly[e];
            const uint32_t pos = beg + atomicAdd(&h[d], 1u);
            p.s_edge[pos] = make_uint2(p.tgt[e] | (p.packed ? d << 24 : 0u), (uint32_t)p.wfx[e]);
            p.s_dly[pos] = (uint8_t)d;
            if (p.plastic) {                                // weights become state: they start at the quantised value
                p.perm[pos] = e;
                p.w_f32[pos] = __fmul_rn(__int2float_rn(p.wfx[e]), 0x1p-16f);
            }
        }
        __syncwarp();
    }
}

// ---- a5: one camera frame -------------------------------------------------------------------------------
// z_j = n * mean(c_j over the frame) + b + gamma * N(0,1).  Box-Muller on the
// vertex group's Philox block: counter {j/4, frame lo, frame hi, 6}; vertices 0,1 use words (x0,x1),
// vertices 2,3 use (x2,x3); even vertex = cosine branch, odd = sine branch.
__global__ void __launch_bounds__(256)
gn_observe_kernel(const GnDev p, const uint64_t frame, const uint32_t trace_row)
{
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    const uint32_t j0 = g * 4u;
    if (j0 >= p.Npad) return;
    const float4 a4 = *reinterpret_cast<const float4 *>(p.acc + j0);
    float z[4] = {0.f, 0.f, 0.f, 0.f};
    if (p.obs_sigma != 0.0f) {
        uint32_t x[4];
        philox4x32_10(g, (uint32_t)frame, (uint32_t)(frame >> 32), kStreamNoise, p.seed_lo, p.seed_hi, x);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const float ua = __fmaf_rn((float)(x[2 * h] >> 9), 0x1p-23f, 0x1p-24f);   // (k + 1/2) 2^-23
            const float ub2 = __fmul_rn((float)(x[2 * h + 1] >> 8), 0x1p-23f);         // 2 * u_b
            const float rad = sqrtf(-2.0f * logf(ua));
            float sn, cs;
            sincospif(ub2, &sn, &cs);
            z[2 * h] = rad * cs;
            z[2 * h + 1] = rad * sn;
        }
    }
    const float acc[4] = {a4.x, a4.y, a4.z, a4.w};
    float out[4];
#pragma unroll
    for (int q = 0; q < 4; ++q)
        out[q] = p.obs_gain * (acc[q] * p.inv_stride) + p.obs_offset + p.obs_sigma * z[q];
    *reinterpret_cast<float4 *>(p.trace + (size_t)trace_row * p.Npad + j0) = make_float4(out[0], out[1], out[2], out[3]);
    *reinterpret_cast<float4 *>(p.acc + j0) = make_float4(0.f, 0.f, 0.f, 0.f);
}

// ---- resident mode: every network lives in one CTA (a1-a5 for configs whose networks have <= 1024 vertices) ----
// The paper's own workload shape is many small networks (N <= 1000).  Here a CTA owns one
// network for a whole gn_step(n) call: thread i <-> vertex i of the network, V/W/r/c/acc/refr in registers, the
// network's whole delay ring in shared memory ([D][blockDim] int32), delivery by shared-memory integer atomics,
// one __syncthreads per step.  No per-step launch, no HBM traffic for state or ring inside the call: only the CSR
// rows of the vertices that fire (L2/HBM), the raster bits and the trace rows.  Same arithmetic, same generator
// layout, same integer ring as the streaming kernels: results are bit-identical.
// Drive words: the Philox block of vertex group j/4 at step t serves 4 vertices, so the CTA computes the blocks
// of its groups for 4 steps at a time into shared memory (one block per thread) instead of one per thread per step.
constexpr int kResidentPhiloxSteps = 4;

template <bool OBS, bool BIAS, bool PACKED, bool CLUSTER, bool HH>
__global__ void __launch_bounds__(1024, 1)
gn_resident_kernel(const GnDev p, const uint64_t t0, const uint32_t n_steps, const uint32_t raster_on)
{
    // CLUSTER: a network is spread over the p.res_cluster CTAs of one thread-block cluster (1,024 vertices each);
    // an event whose target lives in another CTA is a shared-memory atomic through DSMEM, and the per-step barrier
    // is the cluster's.
    extern __shared__ int32_t s_dyn[];
    __shared__ GnClassDev s_cls[GN_MAX_CLASSES];
    __shared__ unsigned long long s_tot[3];                 // spikes, events, kicks of this CTA
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t stride = blockDim.x;
    int32_t *s_ring = s_dyn;                                  // [D][stride]: the ring words of this CTA's vertices
    uint32_t *s_px = reinterpret_cast<uint32_t *>(s_dyn + (size_t)p.D * stride);   // [4 steps][groups][4 words]
    const uint32_t i = threadIdx.x, lane = i & 31u;
    const uint32_t net = CLUSTER ? blockIdx.x / p.res_cluster : blockIdx.x;
    const uint32_t rank = CLUSTER ? blockIdx.x - net * p.res_cluster : 0u;
    const uint32_t v0 = p.net_off[net], nv = p.net_off[net + 1] - v0;      // the network
    const uint32_t c0 = rank * stride;                        // first local vertex of this CTA
    const bool live = c0 + i < nv;
    const uint32_t j = v0 + c0 + i;                           // global vertex id (the caller's)
    const uint32_t c_nv = c0 < nv ? min(stride, nv - c0) : 0u;             // vertices of this CTA
    const uint32_t g0 = (v0 + c0) >> 2, n_groups = c_nv ? ((v0 + c0 + c_nv + 3u) >> 2) - g0 : 0u;

    for (uint32_t q = i; q < p.n_classes * kClassWords; q += stride)   // a CTA may have as few as 32 threads
        reinterpret_cast<uint32_t *>(s_cls)[q] = reinterpret_cast<const uint32_t *>(p.cls_tab)[q];
    if (i < 3u) s_tot[i] = 0ull;
    float V = 0.f, W = 0.f, r = 0.f, c = 0.f, acc = 0.f, U = 0.f, pp = 0.f, gm = 0.f, gh = 0.f;
    uint32_t refr = 0u, cl = 0u;
    if (live) {
        V = p.V[j]; W = p.W[j]; r = p.r[j]; refr = p.refr[j]; cl = p.cls[j];
        if (p.any_alpha) pp = p.p2[j];
        if (HH) { gm = p.hm[j]; gh = p.hh[j]; }
        if (OBS) { c = p.c[j]; acc = p.acc[j]; }
        if (BIAS) U = p.bias[j];
    }
    for (uint32_t s = 0; s < p.D; ++s) s_ring[s * stride + i] = live ? p.ring[(size_t)s * p.Npad + j] : 0;
    if (CLUSTER) cluster.sync(); else __syncthreads();
    const GnClassDev k = s_cls[cl];

    uint32_t slot = (uint32_t)(t0 % p.D);
    uint32_t raster_row = (uint32_t)(t0 % p.raster_rows);
    uint32_t in_frame = OBS ? (uint32_t)(t0 % p.obs_stride) : 0u;        // steps of the current frame already taken
    uint64_t frame = OBS ? t0 / p.obs_stride : 0ull;
    const uint32_t px_off = ((j >> 2) - g0) * 4u + (j & 3u), px_step = n_groups * 4u;
    uint32_t n_spikes = 0u, n_kicks = 0u;
    unsigned long long n_events = 0ull;
    for (uint32_t st = 0; st < n_steps; ++st) {
        const uint64_t t = t0 + st;
        if (p.any_drive && (st % kResidentPhiloxSteps) == 0u) {       // drive words of the next 4 steps
            for (uint32_t q = i; q < n_groups * kResidentPhiloxSteps; q += stride) {
                const uint32_t ks = q / n_groups, gg = q - ks * n_groups;
                const uint64_t tt = t + ks;
                uint32_t x[4];
                philox4x32_10(g0 + gg, (uint32_t)tt, (uint32_t)(tt >> 32), kStreamDrive, p.seed_lo, p.seed_hi, x);
                *reinterpret_cast<uint4 *>(s_px + (size_t)q * 4u) = make_uint4(x[0], x[1], x[2], x[3]);
            }
            __syncthreads();
        }
        // a1: this step's ring word, cleared; Bernoulli kick (reading #12)
        int32_t I = s_ring[slot * stride + i];
        s_ring[slot * stride + i] = 0;
        if (p.any_drive && live) {
            const uint32_t x = s_px[(st % kResidentPhiloxSteps) * px_step + px_off];
            if (x < k.drive_thr) { I += k.kick_fx; ++n_kicks; }
        }
        // a2 + a3
        const bool fired = ((HH && k.hh) ? vertex_step_hh<BIAS>(k, p.dt, I, U, V, W, r, refr, pp, gm, gh)
                                         : vertex_step<BIAS, true>(k, p.dt, I, U, V, W, r, refr, pp)) && live;
        if (OBS) {
            c = __fmaf_rn(p.keep_c, c, fired ? p.ca_jump : 0.0f);            // H_c
            acc = __fadd_rn(acc, c);
        }
        const uint32_t fired_mask = __ballot_sync(0xFFFFFFFFu, fired);
        n_spikes += fired ? 1u : 0u;
        if (raster_on && fired_mask) {                        // rows were zeroed by the launcher; words may straddle CTAs
            const uint32_t jw = j - lane, sh = jw & 31u;
            uint32_t *rowp = p.raster + (size_t)raster_row * p.words_pad + (jw >> 5);
            if (lane == 0u) {
                atomicOr(rowp, fired_mask << sh);
                if (sh && (fired_mask >> (32u - sh))) atomicOr(rowp + 1, fired_mask >> (32u - sh));   // never past the row
            }
        }
        // a4: every fired vertex of the warp in turn, lanes over its row, shared-memory integer atomics
        if (fired_mask) {
            uint32_t beg = 0u, end = 0u;
            if (fired) { beg = p.row[j]; end = p.row[j + 1]; }
            uint32_t m = fired_mask;
            while (m) {
                const uint32_t src_lane = (uint32_t)__ffs(m) - 1u;
                m &= m - 1u;
                const uint32_t b = __shfl_sync(0xFFFFFFFFu, beg, src_lane), e_end = __shfl_sync(0xFFFFFFFFu, end, src_lane);
                for (uint32_t e = b + lane; e < e_end; e += 32u) {
                    const uint2 ev = p.s_edge[e];
                    const uint32_t d = PACKED ? ev.x >> 24 : (uint32_t)p.s_dly[e];
                    const uint32_t tgt = (PACKED ? ev.x & 0xFFFFFFu : ev.x) - v0;     // local vertex of the target
                    uint32_t s = slot + d;
                    if (s >= p.D) s -= p.D;
                    if (CLUSTER) {
                        const uint32_t owner = tgt >> 10;                               // stride is 1,024 in cluster mode
                        atomicAdd(cluster.map_shared_rank(&s_ring[s * stride + (tgt & 1023u)], owner), (int32_t)ev.y);
                    } else {
                        atomicAdd(&s_ring[s * stride + tgt], (int32_t)ev.y);
                    }
                }
                if (lane == 0u) n_events += (unsigned long long)(e_end - b);
            }
        }
        // deliveries must land before the next slot is read: arrive now, wait after the frame work (which touches no ring)
        cg::cluster_group::arrival_token tok;
        if (CLUSTER) tok = cluster.barrier_arrive(); else __syncthreads();
        // a5: camera frame
        if (OBS && ++in_frame == p.obs_stride) {
            float z = 0.f;
            if (p.obs_sigma != 0.0f) {
                uint32_t x[4];
                philox4x32_10(j >> 2, (uint32_t)frame, (uint32_t)(frame >> 32), kStreamNoise, p.seed_lo, p.seed_hi, x);
                const uint32_t h = (j & 3u) >> 1;
                const float ua = __fmaf_rn((float)(x[2 * h] >> 9), 0x1p-23f, 0x1p-24f);
                const float ub2 = __fmul_rn((float)(x[2 * h + 1] >> 8), 0x1p-23f);
                const float rad = sqrtf(-2.0f * logf(ua));
                float sn, cs;
                sincospif(ub2, &sn, &cs);
                z = (j & 1u) ? rad * sn : rad * cs;
            }
            if (live)
                p.trace[(size_t)(frame % p.trace_cap) * p.Npad + j] = p.obs_gain * (acc * p.inv_stride) + p.obs_offset + p.obs_sigma * z;
            acc = 0.f;
            in_frame = 0u;
            ++frame;
        }
        if (CLUSTER) cluster.barrier_wait(std::move(tok));
        if (++slot == p.D) slot = 0u;
        if (++raster_row == p.raster_rows) raster_row = 0u;
    }
    // back to global memory: the state at t0 + n_steps
    if (live) {
        p.V[j] = V; p.W[j] = W; p.r[j] = r; p.refr[j] = (uint8_t)refr;
        if (p.any_alpha) p.p2[j] = pp;
        if (HH) { p.hm[j] = gm; p.hh[j] = gh; }
        if (OBS) { p.c[j] = c; p.acc[j] = acc; }
    }
    for (uint32_t s = 0; s < p.D; ++s)
        if (live) p.ring[(size_t)s * p.Npad + j] = s_ring[s * stride + i];
    n_spikes = __reduce_add_sync(0xFFFFFFFFu, n_spikes);
    n_kicks = __reduce_add_sync(0xFFFFFFFFu, n_kicks);
    if (lane == 0u) {
        if (n_spikes) atomicAdd(&s_tot[0], (unsigned long long)n_spikes);
        if (n_events) atomicAdd(&s_tot[1], n_events);
        if (n_kicks) atomicAdd(&s_tot[2], (unsigned long long)n_kicks);
    }
    __syncthreads();
    if (i == 0u) {
        if (s_tot[0]) atomicAdd(&p.counters[1], s_tot[0]);
        if (s_tot[1]) atomicAdd(&p.counters[2], s_tot[1]);
        if (s_tot[2]) atomicAdd(&p.counters[3], s_tot[2]);
        if (blockIdx.x == 0) p.counters[0] = t0 + n_steps;
    }
}

// ---- persistent step driver for ring-mode networks that fit one co-resident grid (a1-a5) --------
// On a network of up to ~3*10^5 vertices a step is a few microseconds of work, the same order as a kernel launch, so
// one launch per step is bound by launch latency.  Here a whole gn_step(n) call is ONE cooperative launch: thread g
// owns vertices 4g .. 4g+3 for all n steps and keeps their state in registers (V, W, r, p, m, h, c, acc, refr); per
// step it reads and clears its ring words, draws the kicks, advances its vertices, writes its raster nibble, delivers
// the events of its warp's fired vertices (warp-cooperative REDs into the L2-resident ring, as the FUSED update
// kernel) and emits its trace values at a frame boundary; one grid-wide barrier per step makes every delivery visible
// before the slot it lands in is read.  The barrier is split: a CTA ARRIVES as soon as its delay-1 events -- the only
// ones the very next step can read -- are out and fenced, then delivers the rest of its events, does the frame work
// and draws the next step's kicks (none of which the next step's ring read depends on), and only then WAITS; those
// later events are fenced by the arrival of the following step, one step before the earliest slot they touch is read.
// No host call, no launch and no state traffic inside the call.  Same vertex_step, same generator layout, same
// integer ring: bit-identical to the per-step kernels.  `sync` is a device counter that only grows (sync_base = its
// value when the launch starts); a wait that would never end (a bug, never an input) gives up after ~1 s.
template <bool OBS, bool BIAS, bool HH>
__global__ void __launch_bounds__(kUpdateThreads, 2)
gn_persist_kernel(const GnDev p, const uint64_t t0, const uint32_t n_steps, unsigned long long *sync,
                  const unsigned long long sync_base)
{
    __shared__ GnClassDev s_cls[GN_MAX_CLASSES];
    for (uint32_t q = threadIdx.x; q < p.n_classes * kClassWords; q += kUpdateThreads)
        reinterpret_cast<uint32_t *>(s_cls)[q] = reinterpret_cast<const uint32_t *>(p.cls_tab)[q];
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t g = blockIdx.x * kUpdateThreads + threadIdx.x;
    const uint32_t j0 = g * kVertsPerThread;
    const bool mine = j0 < p.Npad;
    float V[4] = {0.f, 0.f, 0.f, 0.f}, W[4] = {0.f, 0.f, 0.f, 0.f}, r[4] = {0.f, 0.f, 0.f, 0.f}, pp[4] = {0.f, 0.f, 0.f, 0.f};
    float gm[4] = {0.f, 0.f, 0.f, 0.f}, gh[4] = {0.f, 0.f, 0.f, 0.f}, c[4] = {0.f, 0.f, 0.f, 0.f}, acc[4] = {0.f, 0.f, 0.f, 0.f};
    float U[4] = {0.f, 0.f, 0.f, 0.f};
    uint32_t refr[4] = {0u, 0u, 0u, 0u}, cl[4] = {0u, 0u, 0u, 0u};
    uint32_t urgent = 0u;                                     // bit q: vertex j0+q has an out-edge of delay 1
    uint32_t rbeg[4] = {0u, 0u, 0u, 0u}, rdeg[4] = {0u, 0u, 0u, 0u};   // row start and out-degree of the thread's vertices (static)
    auto ld4 = [&](const float *a, float (&x)[4]) {
        const float4 v = *reinterpret_cast<const float4 *>(a + j0);
        x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w;
    };
    auto st4 = [&](float *a, const float (&x)[4]) { *reinterpret_cast<float4 *>(a + j0) = make_float4(x[0], x[1], x[2], x[3]); };
    if (mine) {
        ld4(p.V, V); ld4(p.W, W); ld4(p.r, r);
        if (p.any_alpha) ld4(p.p2, pp);
        if (HH) { ld4(p.hm, gm); ld4(p.hh, gh); }
        if (OBS) { ld4(p.c, c); ld4(p.acc, acc); }
        if (BIAS) ld4(p.bias, U);
        const uchar4 rf4 = *reinterpret_cast<const uchar4 *>(p.refr + j0), cl4 = *reinterpret_cast<const uchar4 *>(p.cls + j0);
        refr[0] = rf4.x; refr[1] = rf4.y; refr[2] = rf4.z; refr[3] = rf4.w;
        cl[0] = cl4.x; cl[1] = cl4.y; cl[2] = cl4.z; cl[3] = cl4.w;
        const uchar4 md4 = *reinterpret_cast<const uchar4 *>(p.min_dly + j0);
        urgent = (md4.x == 1u) | ((md4.y == 1u) << 1) | ((md4.z == 1u) << 2) | ((md4.w == 1u) << 3);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            rbeg[q] = p.row[j0 + q];
            rdeg[q] = p.row[j0 + q + 1] - rbeg[q];
        }
    }
    uint32_t slot = (uint32_t)(t0 % p.D), raster_row = (uint32_t)(t0 % p.raster_rows);
    uint32_t in_frame = OBS ? (uint32_t)(t0 % p.obs_stride) : 0u;
    uint64_t frame = OBS ? t0 / p.obs_stride : 0ull;
    uint32_t n_spikes = 0u, n_kicks = 0u;
    unsigned long long n_events = 0ull;
    // bit q: vertex j0+q is kicked at step t (reading #12); drawn one step ahead, behind the barrier
    auto draw_kicks = [&](const uint64_t t) -> uint32_t {
        uint32_t k = 0u;
        if (mine && p.any_drive) {
            uint32_t x[4];
            philox4x32_10(g, (uint32_t)t, (uint32_t)(t >> 32), kStreamDrive, p.seed_lo, p.seed_hi, x);
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if ((j0 + q) < p.N && x[q] < s_cls[cl[q]].drive_thr) k |= 1u << q;
        }
        return k;
    };
    // the edges of the warp's fired vertices (bits of `nib`) with delay == 1 (URGENT) or delay >= 2, lanes over each row
    auto deliver = [&](const uint32_t nib, const bool urgent_pass) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t m = __ballot_sync(0xFFFFFFFFu, (nib >> q) & 1u);
            while (m) {
                const int src_lane = __ffs(m) - 1;
                m &= m - 1u;
                const uint32_t beg = __shfl_sync(0xFFFFFFFFu, rbeg[q], src_lane), deg = __shfl_sync(0xFFFFFFFFu, rdeg[q], src_lane);
                const uint2 *__restrict__ edge = p.s_edge + beg;
                const uint8_t *__restrict__ dly = p.s_dly + beg;
                for (uint32_t x0 = 0u; x0 < deg; x0 += 128u) {          // four 32-edge blocks requested at once
                    uint2 ev[4];
                    uint32_t d[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const uint32_t x = x0 + 32u * u + lane;
                        ev[u] = make_uint2(0u, 0u);
                        d[u] = 0u;
                        if (x < deg) {
                            ev[u] = __ldg(edge + x);
                            d[u] = p.packed ? ev[u].x >> 24 : (uint32_t)__ldg(dly + x);
                        }
                    }
                    bool beyond = false;                                 // urgent pass: an edge with delay > 1 seen (rows are sorted)
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (d[u] == 0u) continue;
                        if ((d[u] == 1u) != urgent_pass) { beyond = true; continue; }
                        uint32_t s1 = slot + d[u];
                        if (s1 >= p.D) s1 -= p.D;
                        atomicAdd(p.ring + (size_t)s1 * p.Npad + (p.packed ? ev[u].x & 0xFFFFFFu : ev[u].x), (int32_t)ev[u].y);
                    }
                    if (urgent_pass && __any_sync(0xFFFFFFFFu, beyond)) break;
                }
                if (!urgent_pass && lane == 0u) n_events += (unsigned long long)deg;
            }
        }
    };
    uint32_t kicks = draw_kicks(t0);
    for (uint32_t st = 0; st < n_steps; ++st) {
        const uint64_t t = t0 + st;
        uint32_t nib = 0u;
        if (mine) {
            int4 *slot_ptr = reinterpret_cast<int4 *>(p.ring + (size_t)slot * p.Npad + j0);
            const int4 I4 = __ldcg(slot_ptr);                 // written by other SMs' REDs: read it where they landed (L2)
            if ((I4.x | I4.y | I4.z | I4.w) != 0) *slot_ptr = make_int4(0, 0, 0, 0);
            int32_t I[4] = {I4.x, I4.y, I4.z, I4.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if ((kicks >> q) & 1u) { I[q] += s_cls[cl[q]].kick_fx; ++n_kicks; }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const GnClassDev &k = s_cls[cl[q]];
                const bool fired = ((HH && k.hh) ? vertex_step_hh<BIAS>(k, p.dt, I[q], U[q], V[q], W[q], r[q], refr[q], pp[q], gm[q], gh[q])
                                                 : vertex_step<BIAS, true>(k, p.dt, I[q], U[q], V[q], W[q], r[q], refr[q], pp[q])) &&
                                   (j0 + q) < p.N;
                if (fired) nib |= 1u << q;
                if (OBS) {
                    c[q] = __fmaf_rn(p.keep_c, c[q], fired ? p.ca_jump : 0.0f);           // H_c
                    acc[q] = __fadd_rn(acc[q], c[q]);
                }
            }
        }
        // a3: raster word (as gn_update_kernel)
        uint32_t word = nib << (4u * (lane & 7u));
        word |= __shfl_xor_sync(0xFFFFFFFFu, word, 1);
        word |= __shfl_xor_sync(0xFFFFFFFFu, word, 2);
        word |= __shfl_xor_sync(0xFFFFFFFFu, word, 4);
        // a4, urgent part: delay-1 events land in the slot the next step reads.  Then ARRIVE at the step's barrier.
        n_spikes += __popc(nib);
        if (__any_sync(0xFFFFFFFFu, (nib & urgent) != 0u)) deliver(nib & urgent, true);
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) atomicAdd(sync, 1ull);
        // a4, the rest, and the raster word: nothing the next step reads
        if ((lane & 7u) == 0u && mine) p.raster[(size_t)raster_row * p.words_pad + (j0 >> 5)] = word;
        if (__any_sync(0xFFFFFFFFu, nib != 0u)) deliver(nib, false);
        // a5: camera frame (as gn_observe_kernel)
        if (OBS && ++in_frame == p.obs_stride) {
            float z[4] = {0.f, 0.f, 0.f, 0.f};
            if (p.obs_sigma != 0.0f) {
                uint32_t x[4];
                philox4x32_10(g, (uint32_t)frame, (uint32_t)(frame >> 32), kStreamNoise, p.seed_lo, p.seed_hi, x);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float ua = __fmaf_rn((float)(x[2 * h] >> 9), 0x1p-23f, 0x1p-24f);
                    const float ub2 = __fmul_rn((float)(x[2 * h + 1] >> 8), 0x1p-23f);
                    const float rad = sqrtf(-2.0f * logf(ua));
                    float sn, cs;
                    sincospif(ub2, &sn, &cs);
                    z[2 * h] = rad * cs;
                    z[2 * h + 1] = rad * sn;
                }
            }
            if (mine) {
                float out[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) out[q] = p.obs_gain * (acc[q] * p.inv_stride) + p.obs_offset + p.obs_sigma * z[q];
                *reinterpret_cast<float4 *>(p.trace + (size_t)(frame % p.trace_cap) * p.Npad + j0) = make_float4(out[0], out[1], out[2], out[3]);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[q] = 0.f;
            in_frame = 0u;
            ++frame;
        }
        kicks = draw_kicks(t + 1ull);
        // WAIT: every CTA has arrived, so every delay-1 event of step t (and every event of the steps before) has landed
        if (threadIdx.x == 0) {
            const unsigned long long target = sync_base + (unsigned long long)(st + 1u) * gridDim.x;
            long long c0 = 0;
            for (uint32_t spins = 0; *reinterpret_cast<volatile unsigned long long *>(sync) < target; ++spins) {
                if (spins == 1024u) c0 = clock64();
                if (spins > 1024u && clock64() - c0 > 2000000000ll) {       // never seen: the grid is co-resident by construction
                    sync[1] = 1ull;                                         // sticky: the host turns it into GN_E_CUDA
                    break;
                }
            }
            __threadfence();
        }
        __syncthreads();
        if (++slot == p.D) slot = 0u;
        if (++raster_row == p.raster_rows) raster_row = 0u;
    }
    if (mine) {
        st4(p.V, V); st4(p.W, W); st4(p.r, r);
        if (p.any_alpha) st4(p.p2, pp);
        if (HH) { st4(p.hm, gm); st4(p.hh, gh); }
        if (OBS) { st4(p.c, c); st4(p.acc, acc); }
        *reinterpret_cast<uchar4 *>(p.refr + j0) = make_uchar4(refr[0], refr[1], refr[2], refr[3]);
    }
    n_kicks = __reduce_add_sync(0xFFFFFFFFu, n_kicks);
    n_spikes = __reduce_add_sync(0xFFFFFFFFu, n_spikes);
    if (lane == 0u) {
        if (n_spikes) atomicAdd(&p.counters[1], (unsigned long long)n_spikes);
        if (n_events) atomicAdd(&p.counters[2], n_events);
        if (n_kicks) atomicAdd(&p.counters[3], (unsigned long long)n_kicks);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) p.counters[0] = t0 + n_steps;
}

// ---- plastic mode: spike-time dependent plasticity (eq. 32-33; readings #22, #23) ----------
// Every weight is a state of its own (eq. 9) and eq. 30 weighs an arriving spike with the weight AT THE ARRIVAL step, so
// nothing is delivered when a vertex fires: per step t
//   gn_arrive_kernel         for every delay d and every vertex i that fired at t - d (the spike list of that step), the edges
//                            of i with delay exactly d -- a contiguous run of its delay-sorted row, boundaries from the
//                            per-delay table (q_seg with groups of one slot) -- add rint(w(t) 2^16) to ring[t mod D][target];
//   gn_update_kernel         as ever (a1-a3); it sends nothing itself;
//   gn_spikes_kernel         the fired vertices of step t, listed (row t mod D of pl_list: the spikes in flight are these
//                            lists), and eq. 32 as integers: row t+1 of ls_hist = t where the vertex fired, else row t;
//   gn_plast_kernel          eq. 33, its two halves in alternate CTAs:
//     (weakening)            the same enumeration again, now that the spikes of step t are known: an arrival at a target
//                            that does not fire at t weakens its edge, w -= dt alpha exp(-beta s_j(t));
//     (strengthening)        every vertex j that fired at t strengthens each in-edge (i -> j, d) on which nothing arrives
//                            at t: w += dt alpha exp(-beta s_i(t - d)), the age read from the history of last-spike steps;
// An edge is touched by at most one thread per step (one arrival per step; weakening needs the target silent,
// strengthening needs it firing), so the weights need no atomics.  Arithmetic (fp32, one rounded operation each):
// age = steps * dt with steps = t - last - 1 (eq. 32: the age is 0 for the step after a spike, so steps = 0 is q = 0: no
// change); dw = (dt alpha) * exp32(-(beta * age)); w +- dw.
template <bool PACKED>
__device__ __forceinline__ uint32_t delay_bound(const GnDev &p, const uint32_t i, const uint32_t d, const uint32_t beg, const uint32_t deg)
{
    // #edges of vertex i with delay < d, 1 <= d <= D: table entry d - 1 of its line (groups of one slot)
    return seg_bound<PACKED>(p, p.q_seg + (size_t)i * p.D, d - 1u, d, beg, deg);
}

__device__ __forceinline__ float stdp_dw(const GnDev &p, const uint32_t steps)
{
    const float age = __fmul_rn(__uint2float_rn(steps), p.dt);
    return __fmul_rn(p.stdp_dta, exp32(-__fmul_rn(p.stdp_beta, age)));
}

// The fired vertices of step t, listed (any order) in row t mod D of pl_list; log_n[t mod D] = how many (zeroed by the
// launcher).  And eq. 32 as integers: row t+1 of ls_hist (D + 1 rows, so that the row of step t - (D-1) survives) = t where
// the vertex fired, else row t.
__global__ void __launch_bounds__(256)
gn_spikes_kernel(const GnDev p, const uint64_t t)
{
    const uint32_t j = blockIdx.x * 256u + threadIdx.x, lane = threadIdx.x & 31u;
    const uint32_t slot = (uint32_t)(t % p.D);
    bool fired = false;
    if (j < p.Npad) {
        fired = (p.raster[(size_t)(t % p.raster_rows) * p.words_pad + (j >> 5)] >> (j & 31u)) & 1u;
        p.ls_hist[(size_t)((t + 1ull) % (p.D + 1u)) * p.Npad + j] = fired ? (int32_t)t : p.ls_hist[(size_t)(t % (p.D + 1u)) * p.Npad + j];
    }
    const uint32_t m = __ballot_sync(0xFFFFFFFFu, fired);
    if (m == 0u) return;
    uint32_t base = 0u;
    if (lane == 0u) {
        base = atomicAdd(&p.log_n[slot], (uint32_t)__popc(m));
        atomicAdd(&p.counters[1], (unsigned long long)__popc(m));
    }
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (fired) p.pl_list[(size_t)slot * p.Npad + base + __popc(m & ((1u << lane) - 1u))] = j;
}

// One thread per (delay d, vertex that fired at t - d), the pairs flattened over the lists of the last n_d steps.
template <bool LTD, bool PACKED>
__device__ __forceinline__ void arrive_body(const GnDev &p, const uint64_t t, const uint32_t n_d, const uint32_t bid, const uint32_t n_blocks)
{
    __shared__ uint32_t s_pref[256];
    __shared__ uint32_t s_wsum[8];
    uint32_t cnt = 0u;
    if (threadIdx.x < n_d) cnt = p.log_n[(t - 1ull - threadIdx.x) % p.D];      // delay d = threadIdx.x + 1
    uint32_t off;
    const uint32_t P = gather_scan<256>(cnt, s_wsum, off);
    s_pref[threadIdx.x] = off;
    __syncthreads();
    unsigned long long events = 0ull;
    const uint32_t slot = (uint32_t)(t % p.D);
    const uint32_t *fired_now = p.raster + (size_t)(t % p.raster_rows) * p.words_pad;
    const int32_t *last = p.ls_hist + (size_t)(t % (p.D + 1u)) * p.Npad;
    for (uint32_t pidx = bid * 256u + threadIdx.x; pidx < P; pidx += n_blocks * 256u) {
        uint32_t lo = 0u, hi_s = n_d;                       // the last delay index whose pairs start at or before pidx
        while (hi_s - lo > 1u) {
            const uint32_t mid = (lo + hi_s) >> 1;
            if (s_pref[mid] <= pidx) lo = mid; else hi_s = mid;
        }
        const uint32_t d = lo + 1u;
        const uint32_t i = p.pl_list[(size_t)((t - d) % p.D) * p.Npad + (pidx - s_pref[lo])];
        const uint32_t beg = p.row[i], deg = p.row[i + 1] - beg;
        const uint32_t e_lo = delay_bound<PACKED>(p, i, d, beg, deg), e_hi = delay_bound<PACKED>(p, i, d + 1u, beg, deg);
        for (uint32_t e = beg + e_lo; e < beg + e_hi; ++e) {
            const uint32_t m = PACKED ? p.s_edge[e].x & 0xFFFFFFu : p.s_edge[e].x;
            if (!LTD) {
                // eq. 33 has no ceiling: unlike a static weight (checked once by gn_create) a plastic one can leave the
                // fixed-point range; the conversion saturates, and the delivery is counted (GN_FAULTS[0])
                const float s = __fmul_rn(p.w_f32[e], 65536.0f);
                ring_add(p.ring + (size_t)slot * p.Npad + m, __float2int_rn(s));
                if (!(fabsf(s) < 2147483648.0f)) atomicAdd(&p.faults[0], 1ull);
            } else if (!((fired_now[m >> 5] >> (m & 31u)) & 1u)) {         // (a coincidence changes nothing)
                const int32_t ls = last[m];
                if (ls >= 0 && (uint64_t)ls + 1ull < t)
                    p.w_f32[e] = __fsub_rn(p.w_f32[e], stdp_dw(p, (uint32_t)(t - 1ull - (uint64_t)ls)));
            }
        }
        events += (unsigned long long)(e_hi - e_lo);
    }
    if (!LTD) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) events += __shfl_xor_sync(0xFFFFFFFFu, events, o);
        if ((threadIdx.x & 31u) == 0u && events) atomicAdd(&p.counters[2], events);
    }
}

// One warp per vertex that fired at t (its list), lanes over its in-edges.
template <bool PACKED>
__device__ __forceinline__ void ltp_body(const GnDev &p, const uint64_t t, const uint32_t bid, const uint32_t n_blocks)
{
    const uint32_t lane = threadIdx.x & 31u, n_warps = (n_blocks * 256u) >> 5;
    const uint32_t slot = (uint32_t)(t % p.D), n = p.log_n[slot];
    for (uint32_t q = (bid * 256u + threadIdx.x) >> 5; q < n; q += n_warps) {
        const uint32_t j = p.pl_list[(size_t)slot * p.Npad + q];
        for (uint32_t k = p.csc_off[j] + lane; k < p.csc_off[j + 1]; k += 32u) {
            const uint32_t e = p.csc_edge[k], i = p.csc_src[k];
            const uint32_t d = PACKED ? p.s_edge[e].x >> 24 : (uint32_t)p.s_dly[e];
            if ((uint64_t)d > t) continue;                 // nothing of i can have arrived yet, and i has no age d steps ago
            const uint64_t td = t - d;
            const uint32_t arr = p.raster[(size_t)(td % p.raster_rows) * p.words_pad + (i >> 5)];
            if ((arr >> (i & 31u)) & 1u) continue;        // the spike of i arrives now: coincidence
            const int32_t ls = p.ls_hist[(size_t)(td % (p.D + 1u)) * p.Npad + i];
            if (ls >= 0 && (uint64_t)ls + 1ull < td)
                p.w_f32[e] = __fadd_rn(p.w_f32[e], stdp_dw(p, (uint32_t)(td - 1ull - (uint64_t)ls)));
        }
    }
}

// Delivery at arrival time (before the update of step t).
template <bool PACKED>
__global__ void __launch_bounds__(256)
gn_arrive_kernel(const GnDev p, const uint64_t t, const uint32_t n_d)
{
    arrive_body<false, PACKED>(p, t, n_d, blockIdx.x, gridDim.x);
}

// eq. 33 (after the update of step t and gn_spikes_kernel): even CTAs weaken at the step's arrivals, odd CTAs strengthen at
// its spikes -- different edges, so the two halves need nothing from each other.
template <bool PACKED>
__global__ void __launch_bounds__(256)
gn_plast_kernel(const GnDev p, const uint64_t t, const uint32_t n_d)
{
    if ((blockIdx.x & 1u) == 0u) {
        if (n_d) arrive_body<true, PACKED>(p, t, n_d, blockIdx.x >> 1, gridDim.x >> 1);
    } else {
        ltp_body<PACKED>(p, t, blockIdx.x >> 1, gridDim.x >> 1);
    }
}

// in-edge lists: count, scan, fill
__global__ void gn_csc_count_kernel(const GnDev p, const uint32_t n_edges, const bool packed)
{
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n_edges) atomicAdd(&p.csc_off[(packed ? p.s_edge[e].x & 0xFFFFFFu : p.s_edge[e].x) + 1u], 1u);
}

__global__ void __launch_bounds__(1024)
gn_csc_scan_kernel(uint32_t *a, const uint32_t n)         // in place, inclusive (a[0] = 0 makes it the offsets); one CTA
{
    __shared__ uint32_t s_w[32];
    __shared__ uint32_t s_carry;
    if (threadIdx.x == 0) s_carry = 0u;
    __syncthreads();
    for (uint32_t b = 0; b < n; b += 1024u) {
        const uint32_t idx = b + threadIdx.x, lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
        uint32_t v = idx < n ? a[idx] : 0u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, v, o);
            if (lane >= (uint32_t)o) v += u;
        }
        if (lane == 31u) s_w[warp] = v;
        __syncthreads();
        uint32_t before = s_carry;
        for (uint32_t k = 0; k < warp; ++k) before += s_w[k];
        if (idx < n) a[idx] = v + before;
        __syncthreads();
        if (threadIdx.x == 1023u) s_carry = v + before;
        __syncthreads();
    }
}

__global__ void gn_csc_fill_kernel(const GnDev p, uint32_t *cursor, const bool packed)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= p.N) return;
    for (uint32_t e = p.row[i] + lane; e < p.row[i + 1]; e += 32u) {
        const uint32_t m = packed ? p.s_edge[e].x & 0xFFFFFFu : p.s_edge[e].x;
        const uint32_t k = p.csc_off[m] + atomicAdd(&cursor[m], 1u);
        p.csc_edge[k] = e;
        p.csc_src[k] = i;
    }
}

__global__ void gn_weights_out_kernel(const GnDev p, const uint32_t n_edges)
{
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n_edges) p.w_stage[p.perm[e]] = p.w_f32[e];
}

// ---- create-time kernels --------------------------------------------------------------------------------
// gn_create's overflow bound (gn_validate_kernel + gn_check_overflow_kernel) over the CURRENT plastic weights: a target
// whose sum of |w_fx| over its in-edges plus its class's kick passes 2^31 - 1 is counted in faults[1].  The sums only
// grow, so the one addition that carries a sum across its limit counts the target, once.  abs_in and faults[1] hold zeros.
__global__ void gn_plastic_headroom_kernel(const GnDev p, const uint32_t n_edges, unsigned long long *abs_in)
{
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_edges) return;
    const uint32_t m = p.packed ? p.s_edge[e].x & 0xFFFFFFu : p.s_edge[e].x;
    const float s = __fmul_rn(p.w_f32[e], 65536.0f);
    const long long w = __float2int_rn(s);
    // a weight outside the fixed-point range (or NaN) counts as 2^31: its target is over the bound whatever else arrives
    const unsigned long long a = !(fabsf(s) < 2147483648.0f) ? 2147483648ull : (unsigned long long)(w < 0 ? -w : w);
    if (a == 0ull) return;
    uint32_t k = p.cls[m];
    if (k >= p.n_classes) k = 0u;
    const long long kick = p.cls_tab[k].kick_fx;
    const unsigned long long limit = 2147483647ull - (unsigned long long)(kick < 0 ? -kick : kick);
    const unsigned long long before = atomicAdd(&abs_in[m], a);
    if (before <= limit && before + a > limit) atomicAdd(&p.faults[1], 1ull);
}

__global__ void gn_init_state_kernel(const GnDev p, GnCheck *chk)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.Npad) return;
    uint32_t k = p.cls[j];
    if (j >= p.N) k = 0u;
    if (k >= p.n_classes) {
        chk->bad_class = 1u;
        k = 0u;
    }
    const GnClassDev &q = p.cls_tab[k];
    p.V[j] = q.hh ? q.hh_v0 : -70.0f;                       // reading #15; Hodgkin-Huxley: at rest, gates at their steady states
    p.W[j] = q.hh ? q.hh_n0 : __fmul_rn(q.b, -70.0f);
    p.hm[j] = q.hh ? q.hh_m0 : 0.0f;
    p.hh[j] = q.hh ? q.hh_h0 : 0.0f;
    p.r[j] = 0.0f;
    p.p2[j] = 0.0f;
    p.refr[j] = 0;
    if (p.c) { p.c[j] = 0.0f; p.acc[j] = 0.0f; }
}

__global__ void gn_convert_rows_kernel(const GnDev p, const uint64_t *row64, const uint64_t n_edges, GnCheck *chk)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > p.Npad) return;
    if (i > p.N) { p.row[i] = (uint32_t)n_edges; return; }
    const uint64_t v = row64[i];
    if (i == 0 && v != 0ull) chk->bad_row = 1u;
    if (i == p.N && v != n_edges) chk->bad_row = 1u;
    if (i < p.N && row64[i + 1] < v) chk->bad_row = 1u;
    if (v > n_edges) chk->bad_row = 1u;
    p.row[i] = (uint32_t)(v > n_edges ? n_edges : v);
}

// w_fx = rint(w * 2^16), ties to even, in place over the fp32 weights (w * 2^16 is exact in binary32).
__global__ void gn_quantise_kernel(const GnDev p, const uint64_t n_edges, GnCheck *chk)
{
    for (uint64_t e = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; e < n_edges; e += (uint64_t)gridDim.x * blockDim.x) {
        const float s = __fmul_rn(__int_as_float(p.wfx[e]), 65536.0f);
        if (!(fabsf(s) < 2147483648.0f)) {                  // also catches NaN
            chk->bad_weight = 1u;
            p.wfx[e] = 0;
        } else {
            p.wfx[e] = __float2int_rn(s);
        }
    }
}

// PAPER.md:251 eq. 25 in steps: max(1, ceil(|x_i - x_j| / (speed * dt))), double, no contraction.
__global__ void gn_delays_kernel(const GnDev p, const float *__restrict__ pos, const uint32_t dim, const float speed,
                                 GnCheck *chk)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= p.N) return;
    const double per_step = __dmul_rn((double)speed, (double)p.dt);
    double xi[3] = {0.0, 0.0, 0.0};
    for (uint32_t k = 0; k < dim; ++k) xi[k] = (double)pos[(size_t)i * dim + k];
    for (uint32_t e = p.row[i] + lane; e < p.row[i + 1]; e += 32u) {
        const uint32_t m = p.tgt[e];
        double d2 = 0.0;
        if (m < p.N) {
            for (uint32_t k = 0; k < dim; ++k) {
                const double d = __dsub_rn(xi[k], (double)pos[(size_t)m * dim + k]);
                d2 = __dadd_rn(d2, __dmul_rn(d, d));
            }
        }
        double steps = ceil(__ddiv_rn(__dsqrt_rn(d2), per_step));
        if (!(d2 < 1e300)) chk->bad_position = 1u;          // NaN or infinite coordinate: no distance, no delay
        if (!(steps >= 1.0)) steps = 1.0;                   // coincident points (reading #7)
        if (steps > 255.0) steps = 255.0;                   // >= D is rejected by the validation kernel
        p.dly[e] = (uint8_t)steps;
    }
}

// Per edge: target range, delay range, same network; per target: sum of |w_fx| (overflow bound).
__global__ void gn_validate_kernel(const GnDev p, const uint32_t *__restrict__ net_offsets, const uint32_t n_networks,
                                   unsigned long long *abs_in, GnCheck *chk)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= p.N) return;
    uint32_t lo_v = 0u, hi_v = p.N;                          // vertex range of i's network
    if (net_offsets) {
        uint32_t lo = 0u, hi = n_networks;                   // find b with net_offsets[b] <= i < net_offsets[b+1]
        while (hi - lo > 1u) {
            const uint32_t mid = (lo + hi) >> 1;
            if (net_offsets[mid] <= i) lo = mid; else hi = mid;
        }
        lo_v = net_offsets[lo];
        hi_v = net_offsets[lo + 1];
    }
    for (uint32_t e = p.row[i] + lane; e < p.row[i + 1]; e += 32u) {
        const uint32_t m = p.tgt[e];
        const uint32_t d = p.dly[e];
        if (d < 1u || d > p.D - 1u) chk->bad_delay = 1u;
        if (m >= p.N) { chk->bad_target = 1u; continue; }
        if (m < lo_v || m >= hi_v) chk->cross_net = 1u;
        const int32_t w = p.wfx[e];
        const unsigned long long a = (unsigned long long)(w < 0 ? -(long long)w : (long long)w);
        if (a) atomicAdd(&abs_in[m], a);
    }
}

__global__ void gn_check_overflow_kernel(const GnDev p, const unsigned long long *__restrict__ abs_in, GnCheck *chk)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.N) return;
    uint32_t k = p.cls[j];
    if (k >= p.n_classes) k = 0u;
    const long long kick = p.cls_tab[k].kick_fx;
    const unsigned long long bound = abs_in[j] + (unsigned long long)(kick < 0 ? -kick : kick);
    if (bound > 2147483647ull) chk->overflow = 1u;
}

__global__ void gn_debug_words_kernel(const uint32_t seed_lo, const uint32_t seed_hi, const uint32_t stream_id,
                                      const uint64_t idx, const uint32_t first, const uint32_t n, uint32_t *out)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t j = first + i;
    uint32_t x[4];
    philox4x32_10(j >> 2, (uint32_t)idx, (uint32_t)(idx >> 32), stream_id, seed_lo, seed_hi, x);
    out[i] = x[j & 3u];
}

// ---- measured ceilings of the delivery pattern (gn_debug_ceilings: the roofline bench.py rates a4 against) -----------
// Scattered int32 reductions into a region of `mask + 1` words that stays in L2 -- and the same preceded by the gather of
// the 8-byte edge each reduction carries, read in random contiguous segments of seg_len edges (unaligned starts) from an
// array far larger than L2, 32 edges per load instruction, four loads in flight per warp: the access pattern of
// gn_fold_kernel with everything else stripped off.
__device__ __forceinline__ uint32_t ceil_mix(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

template <bool GATHER>
__global__ void __launch_bounds__(256)
gn_ceiling_kernel(int32_t *region, const uint32_t mask, const uint2 *edges, const uint32_t n_edges, const uint32_t seg_len,
                  const uint32_t iters, const uint32_t seed)
{
    const uint32_t lane = threadIdx.x & 31u, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    for (uint32_t it = 0; it < iters; it += 4u) {
        uint2 e[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t slot = (it + u) * 32u + lane;
            if (GATHER) {
                const uint32_t seg = slot / seg_len, k = slot - seg * seg_len;
                const uint32_t start = ceil_mix(gw * 0x9E3779B9u + seg * 0x85EBCA6Bu + seed) % (n_edges - seg_len);
                e[u] = __ldcs(edges + start + k);
                e[u].x ^= ceil_mix(slot + gw);
            } else {
                e[u] = make_uint2(ceil_mix(ceil_mix(gw * 0x9E3779B9u + seed) + slot), 1u);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) ring_add(region + (e[u].x & mask), (int32_t)e[u].y);
    }
}

inline uint32_t ceil_div(uint64_t a, uint64_t b) { return (uint32_t)((a + b - 1) / b); }

}  // namespace

// ---- launchers ------------------------------------------------------------------------------------------
cudaError_t gnk_update(const GnDev &p, uint64_t t, bool has_bias, cudaStream_t st)
{
    // delays below d_direct are delivered by the update kernel itself (see the kernel)
    const uint32_t d_direct = p.plastic ? 1u      // plastic mode: nothing is sent when a vertex fires (delivery happens at arrival)
                            : p.queue_mode ? (p.q_window << p.q_log) - ((uint32_t)(t % p.D) & ((1u << p.q_log) - 1u)) : 2u;
    const uint32_t grid = ceil_div(p.Npad / kVertsPerThread, kUpdateThreads);
    const uint32_t slot = (uint32_t)(t % p.D);
    const uint32_t raster_row = (uint32_t)(t % p.raster_rows);
    const bool obs = p.obs_stride != 0u;
    // programmatic stream serialization: this launch may begin (up to its griddepcontrol.wait) while the previous
    // kernel in the stream -- normally the previous step's update -- is still draining
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kUpdateThreads);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define GN_UPD2(O, B, A, H)                                                                                      \
    return p.fused ? cudaLaunchKernelEx(&cfg, gn_update_kernel<O, B, true, A, H>, p, t, slot, raster_row, d_direct)  \
                   : cudaLaunchKernelEx(&cfg, gn_update_kernel<O, B, false, A, H>, p, t, slot, raster_row, d_direct)
#define GN_UPD(O, B)                                                                                              \
    do {                                                                                                          \
        if (p.any_hh) GN_UPD2(O, B, true, true);      /* a Hodgkin-Huxley network: one variant for either PSC */     \
        if (p.any_alpha) GN_UPD2(O, B, true, false);                                                              \
        GN_UPD2(O, B, false, false);                                                                              \
    } while (0)
    if (obs && has_bias) GN_UPD(true, true);
    if (obs) GN_UPD(true, false);
    if (has_bias) GN_UPD(false, true);
    GN_UPD(false, false);
#undef GN_UPD2
#undef GN_UPD
}

typedef void (*PersistKernel)(const GnDev, const uint64_t, const uint32_t, unsigned long long *, const unsigned long long);

static PersistKernel persist_kernel_for(const GnDev &p, bool has_bias)
{
    const bool obs = p.obs_stride != 0u;
    if (p.any_hh) return obs ? (has_bias ? gn_persist_kernel<true, true, true> : gn_persist_kernel<true, false, true>)
                             : (has_bias ? gn_persist_kernel<false, true, true> : gn_persist_kernel<false, false, true>);
    return obs ? (has_bias ? gn_persist_kernel<true, true, false> : gn_persist_kernel<true, false, false>)
               : (has_bias ? gn_persist_kernel<false, true, false> : gn_persist_kernel<false, false, false>);
}

// Can the whole grid of the persistent step driver be co-resident on this device (a cooperative launch needs it)?
cudaError_t gnk_persist_ok(const GnDev &p, bool *ok)
{
    *ok = false;
    int dev = 0, coop = 0, sms = 0, per_sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // the variant with the largest footprint decides for all of them
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gn_persist_kernel<true, true, true>, kUpdateThreads, 0);
    if (e != cudaSuccess) { cudaGetLastError(); return cudaSuccess; }
    *ok = coop && (uint64_t)ceil_div(p.Npad / kVertsPerThread, kUpdateThreads) <= (uint64_t)sms * (uint64_t)per_sm;
    return cudaSuccess;
}

cudaError_t gnk_persist(const GnDev &p, uint64_t t0, uint32_t n_steps, bool has_bias, unsigned long long *sync,
                        unsigned long long *sync_base, cudaStream_t st)
{
    GnDev pv = p;
    uint64_t t = t0;
    uint32_t n = n_steps;
    unsigned long long base = *sync_base;
    void *args[5] = {&pv, &t, &n, &sync, &base};
    *sync_base += (unsigned long long)n_steps * ceil_div(p.Npad / kVertsPerThread, kUpdateThreads);   // where the counter ends
    return cudaLaunchCooperativeKernel((const void *)persist_kernel_for(p, has_bias),
                                       dim3(ceil_div(p.Npad / kVertsPerThread, kUpdateThreads)), dim3(kUpdateThreads), args, 0, st);
}

typedef void (*ResidentKernel)(const GnDev, const uint64_t, const uint32_t, const uint32_t);

static cudaError_t resident_config(ResidentKernel k, const GnDev &p, cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr)
{
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.res_smem);
    if (e == cudaSuccess && p.res_cluster > 8u) e = cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(p.n_networks * p.res_cluster);
    cfg.blockDim = dim3(p.res_threads);
    cfg.dynamicSmemBytes = p.res_smem;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = p.res_cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.res_cluster > 1u ? 1 : 0;
    return e;
}

static cudaError_t resident_launch(ResidentKernel k, const GnDev &p, uint64_t t0, uint32_t n_steps, bool raster_on, cudaStream_t st)
{
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cudaError_t e = resident_config(k, p, cfg, attr);
    if (e != cudaSuccess) return e;
    cfg.stream = st;
    return cudaLaunchKernelEx(&cfg, k, p, t0, n_steps, raster_on ? 1u : 0u);
}

// Can the device co-schedule a cluster of p.res_cluster CTAs of the resident kernel at all?
cudaError_t gnk_resident_cluster_ok(const GnDev &p, bool *ok)
{
    *ok = true;
    if (p.res_cluster <= 1u) return cudaSuccess;
    ResidentKernel k = p.packed ? gn_resident_kernel<false, false, true, true, false> : gn_resident_kernel<false, false, false, true, false>;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cudaError_t e = resident_config(k, p, cfg, attr);
    int n = 0;
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(&n, k, &cfg);
    *ok = (e == cudaSuccess && n > 0);
    cudaGetLastError();
    return cudaSuccess;
}

// Resident mode: one CTA (or one cluster) per network for n_steps steps.  Raster rows of these steps are zeroed first (the kernel ORs bits
// into words that may straddle two networks); the caller keeps n_steps <= raster_rows when a raster is kept.
cudaError_t gnk_resident(const GnDev &p, uint64_t t0, uint32_t n_steps, bool has_bias, bool raster_on, cudaStream_t st)
{
    if (raster_on) {
        const uint32_t r0 = (uint32_t)(t0 % p.raster_rows);
        const uint32_t first = n_steps < p.raster_rows - r0 ? n_steps : p.raster_rows - r0;
        cudaError_t e = cudaMemsetAsync(p.raster + (size_t)r0 * p.words_pad, 0, (size_t)first * p.words_pad * 4, st);
        if (e == cudaSuccess && first < n_steps)
            e = cudaMemsetAsync(p.raster, 0, (size_t)(n_steps - first) * p.words_pad * 4, st);
        if (e != cudaSuccess) return e;
    }
    const bool obs = p.obs_stride != 0u;
#define GN_RES_LAUNCH2(O, B, P, H)                                                                               \
    do {                                                                                                        \
        if (p.res_cluster > 1u) return resident_launch(gn_resident_kernel<O, B, P, true, H>, p, t0, n_steps, raster_on, st);  \
        return resident_launch(gn_resident_kernel<O, B, P, false, H>, p, t0, n_steps, raster_on, st);              \
    } while (0)
#define GN_RES_LAUNCH(O, B, P)                                                                                  \
    do {                                                                                                        \
        if (p.any_hh) GN_RES_LAUNCH2(O, B, P, true);                                                            \
        GN_RES_LAUNCH2(O, B, P, false);                                                                         \
    } while (0)
    if (p.packed) {
        if (obs && has_bias) GN_RES_LAUNCH(true, true, true);
        if (obs) GN_RES_LAUNCH(true, false, true);
        if (has_bias) GN_RES_LAUNCH(false, true, true);
        GN_RES_LAUNCH(false, false, true);
    }
    if (obs && has_bias) GN_RES_LAUNCH(true, true, false);
    if (obs) GN_RES_LAUNCH(true, false, false);
    if (has_bias) GN_RES_LAUNCH(false, true, false);
    GN_RES_LAUNCH(false, false, false);
#undef GN_RES_LAUNCH2
#undef GN_RES_LAUNCH
}

// Raster words per delivery CTA: enough CTAs to fill the chip, at most kMaxChunkWords words each.
static uint32_t chunk_words_for(const GnDev &p, uint32_t resident_ctas)
{
    uint32_t w = ceil_div(p.words_pad, resident_ctas);
    if (w < 4u) w = 4u;
    if (w > kMaxChunkWords) w = kMaxChunkWords;
    return w;
}

cudaError_t gnk_deliver(const GnDev &p, uint64_t t, cudaStream_t st)
{
    const uint32_t w = chunk_words_for(p, 148u * 8u);
    gn_deliver_kernel<<<ceil_div(p.words_pad, w), kDeliverThreads, 0, st>>>(p, (uint32_t)(t % p.D),
                                                                          (uint32_t)(t % p.raster_rows), w);
    return cudaGetLastError();
}

cudaError_t gnk_log(const GnDev &p, uint64_t t0, uint32_t n_batch, uint32_t zero_next, cudaStream_t st)
{
    if (n_batch == 0u) return cudaSuccess;
    const uint32_t slot0 = (uint32_t)(t0 % p.D), row0 = (uint32_t)(t0 % p.raster_rows);
    const uint32_t grid = n_batch * ceil_div(p.words_pad, kLogWarps * 32u);   // a warp per step and 32 raster words
    if (p.packed) gn_log_kernel<true><<<grid, kLogWarps * 32, 0, st>>>(p, slot0, row0, n_batch, zero_next);
    else gn_log_kernel<false><<<grid, kLogWarps * 32, 0, st>>>(p, slot0, row0, n_batch, zero_next);
    return cudaGetLastError();
}

cudaError_t gnk_fold(const GnDev &p, uint64_t t_win, uint32_t n_win, uint64_t g_fold, bool beside_previous, cudaStream_t st)
{
    if (p.q_arrays < 2u || n_win == 0u) return cudaSuccess;      // nothing logged that is due in this group
    const uint32_t win_slot0 = (uint32_t)(t_win % p.D), r_win = (uint32_t)(t_win & ((1ull << p.q_log) - 1ull));
    const uint32_t j_first = (uint32_t)(g_fold - (t_win >> p.q_log));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(148u * (uint32_t)kFoldCtasPerSm);
    cfg.blockDim = dim3(kRouteThreads);
    cfg.stream = st;
    // programmatic stream serialization: the fold may start while the kernel in front of it in the stream (the logging
    // kernel of the same launch, which it does not depend on) is still running
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = beside_previous ? 1 : 0;
    return p.packed ? cudaLaunchKernelEx(&cfg, gn_fold_kernel<true>, p, win_slot0, n_win, r_win, j_first)
                    : cudaLaunchKernelEx(&cfg, gn_fold_kernel<false>, p, win_slot0, n_win, r_win, j_first);
}

// plastic mode: in-edge lists.  csc_off and cursor ([N] words of scratch) hold zeros on entry.
cudaError_t gnk_build_csc(const GnDev &p, uint64_t n_edges, uint32_t *cursor, cudaStream_t st)
{
    if (n_edges) gn_csc_count_kernel<<<ceil_div(n_edges, 256), 256, 0, st>>>(p, (uint32_t)n_edges, p.packed != 0u);
    gn_csc_scan_kernel<<<1, 1024, 0, st>>>(p.csc_off, p.Npad + 1u);
    if (n_edges) gn_csc_fill_kernel<<<ceil_div((uint64_t)p.N * 32, 256), 256, 0, st>>>(p, cursor, p.packed != 0u);
    return cudaGetLastError();
}

// plastic mode, before update(t): the spikes arriving at step t (fired at t - d, d = 1 .. min(D - 1, t - t_origin)) are
// added to ring row t mod D with the weights of step t
cudaError_t gnk_arrive(const GnDev &p, uint64_t t, uint64_t t_origin, cudaStream_t st)
{
    const uint64_t back = t - t_origin;
    const uint32_t n_d = (uint32_t)(back < p.D - 1u ? back : p.D - 1u);
    if (n_d == 0u) return cudaSuccess;
    if (p.packed) gn_arrive_kernel<true><<<148u * 8u, 256, 0, st>>>(p, t, n_d);
    else gn_arrive_kernel<false><<<148u * 8u, 256, 0, st>>>(p, t, n_d);
    return cudaGetLastError();
}

// plastic mode, after update(t): the step's spike list and eq. 32, then eq. 33 for the arrivals and the spikes of step t
cudaError_t gnk_plasticity(const GnDev &p, uint64_t t, uint64_t t_origin, cudaStream_t st)
{
    const uint64_t back = t - t_origin;
    const uint32_t n_d = (uint32_t)(back < p.D - 1u ? back : p.D - 1u);
    cudaError_t e = cudaMemsetAsync(p.log_n + (t % p.D), 0, 4, st);
    if (e != cudaSuccess) return e;
    gn_spikes_kernel<<<ceil_div(p.Npad, 256), 256, 0, st>>>(p, t);
    if (p.packed) gn_plast_kernel<true><<<148u * 16u, 256, 0, st>>>(p, t, n_d);
    else gn_plast_kernel<false><<<148u * 16u, 256, 0, st>>>(p, t, n_d);
    return cudaGetLastError();
}

cudaError_t gnk_weights_out(const GnDev &p, uint64_t n_edges, cudaStream_t st)
{
    if (n_edges) gn_weights_out_kernel<<<ceil_div(n_edges, 256), 256, 0, st>>>(p, (uint32_t)n_edges);
    return cudaGetLastError();
}

cudaError_t gnk_plastic_headroom(const GnDev &p, uint64_t n_edges, unsigned long long *abs_in, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(abs_in, 0, (size_t)p.N * 8, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(p.faults + 1, 0, 8, st);
    if (e != cudaSuccess) return e;
    if (n_edges) gn_plastic_headroom_kernel<<<ceil_div(n_edges, 256), 256, 0, st>>>(p, (uint32_t)n_edges, abs_in);
    return cudaGetLastError();
}

cudaError_t gnk_sort_rows(const GnDev &p, GnCheck *chk, cudaStream_t st)
{
    uint32_t grid = ceil_div((uint64_t)p.N * 32, 256);
    if (grid > 148u * 8u) grid = 148u * 8u;
    gn_sort_rows_kernel<<<grid, 256, 0, st>>>(p, chk);
    return cudaGetLastError();
}

cudaError_t gnk_observe(const GnDev &p, uint64_t frame, cudaStream_t st)
{
    gn_observe_kernel<<<ceil_div(p.Npad / 4, 256), 256, 0, st>>>(p, frame, (uint32_t)(frame % p.trace_cap));
    return cudaGetLastError();
}

cudaError_t gnk_init_state(const GnDev &p, GnCheck *chk, cudaStream_t st)
{
    gn_init_state_kernel<<<ceil_div(p.Npad, 256), 256, 0, st>>>(p, chk);
    return cudaGetLastError();
}

cudaError_t gnk_convert_rows(const GnDev &p, const uint64_t *row64, uint64_t n_edges, GnCheck *chk, cudaStream_t st)
{
    gn_convert_rows_kernel<<<ceil_div((uint64_t)p.Npad + 1, 256), 256, 0, st>>>(p, row64, n_edges, chk);
    return cudaGetLastError();
}

cudaError_t gnk_quantise(const GnDev &p, uint64_t n_edges, GnCheck *chk, cudaStream_t st)
{
    if (n_edges == 0) return cudaSuccess;
    uint32_t grid = ceil_div(n_edges, 256);
    if (grid > 148u * 32u) grid = 148u * 32u;
    gn_quantise_kernel<<<grid, 256, 0, st>>>(p, n_edges, chk);
    return cudaGetLastError();
}

cudaError_t gnk_delays_from_positions(const GnDev &p, const float *pos, uint32_t dim, float speed, GnCheck *chk, cudaStream_t st)
{
    gn_delays_kernel<<<ceil_div((uint64_t)p.N * 32, 256), 256, 0, st>>>(p, pos, dim, speed, chk);
    return cudaGetLastError();
}

cudaError_t gnk_validate(const GnDev &p, const uint32_t *net_offsets, uint32_t n_networks,
                         unsigned long long *abs_in, GnCheck *chk, cudaStream_t st)
{
    gn_validate_kernel<<<ceil_div((uint64_t)p.N * 32, 256), 256, 0, st>>>(p, net_offsets, n_networks, abs_in, chk);
    return cudaGetLastError();
}

cudaError_t gnk_check_overflow(const GnDev &p, const unsigned long long *abs_in, GnCheck *chk, cudaStream_t st)
{
    gn_check_overflow_kernel<<<ceil_div(p.N, 256), 256, 0, st>>>(p, abs_in, chk);
    return cudaGetLastError();
}

cudaError_t gnk_debug_words(uint64_t seed, uint32_t stream_id, uint64_t idx, uint32_t first, uint32_t n,
                            uint32_t *out, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    gn_debug_words_kernel<<<ceil_div(n, 256), 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), stream_id, idx, first, n, out);
    return cudaGetLastError();
}

// out[0] = scattered reductions per second into a 16 MB region; out[1] = gathers of seg_len-edge segments + reductions
// per second.  `scratch` (>= 64 MB + 256 MB; the larger the better: the edge array should dwarf L2) is overwritten.
// Best of 5 launches each, timed with CUDA events on `st`; synchronises.
// Streaming read-modify-write of `n4` float4 words, `passes` times over: with a buffer that fits L2 every pass after the
// first is served by L2 (the update kernel's situation when its state stays resident between steps); with one far larger
// than L2 every pass goes to HBM.  128-bit accesses, consecutive threads on consecutive words, like the update kernel's.
__global__ void __launch_bounds__(256)
gn_stream_ceiling_kernel(float4 *x, const uint32_t n4, const uint32_t passes)
{
    for (uint32_t pass = 0; pass < passes; ++pass)
        for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n4; i += gridDim.x * 256u) {
            float4 v = x[i];
            v.x += 1.0f; v.y += 1.0f; v.z += 1.0f; v.w += 1.0f;
            x[i] = v;
        }
}

cudaError_t gnk_stream_ceilings(void *scratch, size_t scratch_bytes, double out[2], cudaStream_t st)
{
    if (scratch_bytes < (1024u << 20)) return cudaErrorInvalidValue;
    cudaError_t e = cudaMemsetAsync(scratch, 0, scratch_bytes, st);
    cudaEvent_t e0, e1;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    const uint32_t grid = 148u * 8u;
    for (int mode = 0; mode < 2 && e == cudaSuccess; ++mode) {
        const size_t bytes = mode == 0 ? (size_t)(32u << 20) : (scratch_bytes & ~(size_t)4095);
        const uint32_t passes = mode == 0 ? 32u : 2u;
        size_t n4 = bytes / 16;
        if (n4 > 0xFFFF0000ull) n4 = 0xFFFF0000ull;
        float best = 1e30f;
        for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {     // rep 0 also warms L2 for mode 0
            cudaEventRecord(e0, st);
            gn_stream_ceiling_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<float4 *>(scratch), (uint32_t)n4, passes);
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        out[mode] = 2.0 * 16.0 * (double)n4 * passes / ((double)best * 1e-3);     // bytes read + bytes written per second
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}

cudaError_t gnk_ceilings(void *scratch, size_t scratch_bytes, uint32_t seg_len, double out[2], cudaStream_t st)
{
    const size_t region_bytes = 16u << 20;
    if (scratch_bytes < (64u << 20) + (256u << 20) || seg_len == 0u) return cudaErrorInvalidValue;
    int32_t *region = reinterpret_cast<int32_t *>(scratch);
    const uint2 *edges = reinterpret_cast<const uint2 *>(reinterpret_cast<uint8_t *>(scratch) + (64u << 20));
    size_t n_edges = (scratch_bytes - (64u << 20)) / 8;
    if (n_edges > 0xFFFFFF00ull) n_edges = 0xFFFFFF00ull;
    cudaError_t e = cudaMemsetAsync(scratch, 1, scratch_bytes, st);
    cudaEvent_t e0, e1;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    const uint32_t grid = 148u * 8u, iters = 64u, mask = (uint32_t)(region_bytes / 4 - 1);
    const double n = (double)grid * 256.0 * iters;
    for (int mode = 0; mode < 2 && e == cudaSuccess; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 5 && e == cudaSuccess; ++rep) {
            cudaEventRecord(e0, st);
            if (mode == 0) gn_ceiling_kernel<false><<<grid, 256, 0, st>>>(region, mask, edges, (uint32_t)n_edges, seg_len, iters, 7919u * rep);
            else gn_ceiling_kernel<true><<<grid, 256, 0, st>>>(region, mask, edges, (uint32_t)n_edges, seg_len, iters, 7919u * rep);
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (ms < best) best = ms;
        }
        out[mode] = n / ((double)best * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}
