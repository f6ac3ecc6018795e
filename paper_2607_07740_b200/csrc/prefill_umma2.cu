// prefill_umma2.cu -- tcgen05 UMMA bifocal / causal prefill, two query tiles per CTA (bf16, head_dim 128; steps a3-a8, a10).
//
// One CTA PAIR (cluster of 2, tcgen05 cta_group::2) owns 256 query rows (two 128-row tiles) x 2 query heads of one KV
// group: CTA c owns head h0 + c, every UMMA is M = 256 across the pair, and each CTA stages -- and on remote visits
// rotates (Eq.(6)) -- only its half of every K tile.  Each staged / rotated K tile feeds BOTH query tiles, so a
// rotated key serves 512 (row, head) pairs with no exchange between CTAs beyond the pair's shared B operand, and the
// rotation per unit of tensor work is half that of one tile per CTA (prefill_umma.cu).
//   warps 0-3    rotate group: forwards local K stages; on remote visits rotates its K half in shared memory between the
//                TMA load and the MMA; once per CTA it replaces Q in shared memory by Q' = R(Delta q) Q (Eq.(6)), in place
//   warps 4-7    softmax group of tile 0, warps 8-11 of tile 1: ONE thread per query row (no row-max exchange), S loaded once
//                into registers, online softmax with lazy rescaling, epilogue
//   warp 12      K (and Q) TMA producer, warp 13 V TMA producer, warp 15 MMA issuer (leader CTA) / V forwarder (peer CTA)
// TMEM (512 columns): S0 | S1 | O0 | O1.  P_t (bf16) aliases columns 0..63 of S_t.  Tensor-pipe order in steady state:
// P0 V(m), Q0 K(m+1), P1 V(m), Q1 K(m+1): the softmax of one tile runs under the two MMAs of the other.
// Q lives in shared memory (UMMA A operand, SWIZZLE_128B), so the register file is split with setmaxnreg:
// softmax groups 176, rotate group 112, producers / issuer 48.
//
// Visit order per pair: the local visits of either tile (from the upper tile's diagonal down to the lower tile's
// window edge), then the Q -> Q' switch, then the remote visits.  A tile takes part in a visit only when the key tile is
// in its own list (Plan); the straddle tile is visited twice with complementary masks.  All visits of a tile feed ONE
// running (m, l, O) per row: the additive form of the Eq.(7) merge.
#include <cuda.h>
#include <math.h>
#include <type_traits>

#include "common.cuh"
#include "umma.cuh"
#include "rot.cuh"
#include "prefill_v2.cuh"

namespace jetlong {

namespace {

using namespace ptx;
using namespace dev;

constexpr int D = 128, BM = 128, BN = 128;
constexpr int NKMAX = 6, NVMAX = 6;
constexpr int KH_BYTES = 64 * D * 2;                  // this CTA's 64 keys: two 8 KB SWIZZLE_128B boxes (ch 0-63 | 64-127)
constexpr int KBOX = 64 * 128;
constexpr int VH_BYTES = BN * 64 * 2;                 // this CTA's 64 channels of 128 keys
constexpr int QBOX = BM * 128;                        // one Q box: 128 rows x 64 channels
constexpr int QT_BYTES = 2 * QBOX;                    // one Q tile
constexpr int Q_BYTES = 2 * QT_BYTES;                 // both tiles
constexpr int BARS_BYTES = 2048;
constexpr int SMEM_BYTES = 232448;                    // the 227 KB opt-in maximum
constexpr int RING_BYTES = SMEM_BYTES - 1024 /*align slack*/ - Q_BYTES - BARS_BYTES;   // cross-term Q operands + K ring + V ring
constexpr int NTHREADS = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr int POLY_OF_4 = 0;                          // of every 4 exponential pairs, this many use the FMA-pipe polynomial
constexpr int W_SOFTMAX = 4, W_KLOAD = 12, W_VLOAD = 13, W_MMA = 15;   // warps 0-3 rotate, 4-7 / 8-11 softmax of tile 0 / 1
constexpr uint32_t TM_S = 0, TM_O = 256;
// setmaxnreg.inc draws only on what other warps of the CTA released (registers left unallocated at launch are not in the
// pool): the split must balance against 4 warpgroups x 128, or the last group to grow waits forever
constexpr int REGS_ROT = 112, REGS_SOFTMAX = 160, REGS_MISC = 80;
static_assert(REGS_ROT + 2 * REGS_SOFTMAX + REGS_MISC == 512, "register file split");

// ---- optional cycle trace of one CTA (build with -DJL_TRACE; read back with jetlong_debug_trace) ----------------
#ifdef JL_TRACE
constexpr int TR_M = 192, TR_SLOTS = 8, TR_ROLES = 5;     // roles: 0 MMA, 1 softmax tile 0, 2 softmax tile 1, 3 rotate, 4 K producer
__device__ long long g_trace[TR_ROLES * TR_M * TR_SLOTS];
__device__ int g_trace_block = 0;
#define TR(role, m, slot)                                                                                      \
    do {                                                                                                       \
        if (blockIdx.x == g_trace_block && (threadIdx.x & 31) == 0 && (m) >= 0 && (m) < TR_M)                  \
            g_trace[((role) * TR_M + (m)) * TR_SLOTS + (slot)] = clock64();                                    \
    } while (0)
#else
#define TR(role, m, slot) do {} while (0)
#endif

struct Bars {
    uint64_t k_full[NKMAX];    // local: TMA bytes of this CTA's K half landed
    uint64_t k_ready[NKMAX];   // leader: both rotate groups are done with K stage s (8 warp arrivals)
    uint64_t k_empty[NKMAX];   // both: every Q K^T reading K stage s has completed (multicast commit)
    uint64_t v_full[NVMAX];    // local: TMA bytes of this CTA's V half landed
    uint64_t v_ready[NVMAX];   // leader: the other CTA's V half has landed (its forwarding warp)
    uint64_t v_empty[NVMAX];   // both: every P V reading V stage s has completed
    uint64_t s_full[2];        // both: S_t holds Q_t K^T of a visit
    uint64_t p_half[2];        // leader: the first 64 columns of P_t are written (8 warp arrivals): the first half of P V may start
    uint64_t p_full[2];        // leader: both softmax groups of tile t wrote P_t and are done reading S_t (8 warp arrivals)
    uint64_t pv_done[2];       // both: O_t += P_t V of a visit has completed
    uint64_t o_full;           // both: all MMAs done
    uint64_t q_full;           // local: TMA bytes of this CTA's Q tiles landed
    uint64_t q_ready;          // leader: Q landed in both CTAs (8 warp arrivals)
    uint64_t q_local_done;     // both: the last local Q K^T has completed, Q may be overwritten by Q'
    uint64_t q_rot_done;       // leader: Q' staged in both CTAs (8 warp arrivals)
    uint32_t tmem_base;
};
static_assert(sizeof(Bars) <= BARS_BYTES, "Bars");

struct Ring {
    int n, s;
    uint32_t ph;
    __device__ Ring(int n_) : n(n_), s(0), ph(0) {}
    __device__ __forceinline__ void next() { if (++s == n) { s = 0; ph ^= 1u; } }
};

struct Params {
    __nv_bfloat16* out;
    float* lse;
    long long L, w0, G;
    int H_q, H_kv, g;
    int bifocal, precise, prerot, window_only, qk_f16, out_f32;
    int n_qb, n_sb, n_s4;                            // n_sb / n_s4: one past the top 256- / 512-row block of this launch
    const float2* lo;
    const float2* hi;
    const uint32_t* selinfo;
};

struct Visit { int kt; int mode; };                   // mode 0 = causal/control, 1 = local, 2 = remote

// visit list of ONE 128-row query tile qb (step a3): local key tiles [kt_lo, qb] descending, then remote [0, kt_hi] descending
// window_only: 0 = the full bifocal rule; 1 = only the local band 0 <= q-k <= w0 on the stored operands (call A of the
// unfused baseline); 2 = the same band scored with the REMOTE operands (call C: "sliding window, remote q/k"):
// no local visit, the remote list covers the band's key tiles and carries the band's mask
struct Plan {
    int qb, kt_lo, kt_hi, kt_rlo, n_local, n_remote, nv;
    __device__ Plan() : qb(0), kt_lo(1), kt_hi(-1), kt_rlo(0), n_local(0), n_remote(0), nv(0) {}
    __device__ Plan(int qb_, long long w0, bool bifocal, int window_only) : qb(qb_), kt_rlo(0) {
        const long long q0 = (long long)qb * BM;
        if (!bifocal) { kt_lo = 0; n_local = qb + 1; n_remote = 0; kt_hi = -1; nv = n_local; return; }
        long long t = q0 - w0 - (BN - 1);                              // local iff k0 >= t
        kt_lo = t <= 0 ? 0 : (int)((t + BN - 1) / BN);
        n_local = qb - kt_lo + 1;
        long long u = q0 + (BM - 1) - 1 - w0;                          // remote iff k0 <= u  (q0+127-k0 > w0)
        kt_hi = u < 0 ? -1 : (int)(u / BN);
        if (kt_hi > qb) kt_hi = qb;
        if (window_only == 1) kt_hi = -1;
        if (window_only == 2) { kt_rlo = kt_lo; kt_hi = qb; kt_lo = qb + 1; n_local = 0; }
        n_remote = kt_hi - kt_rlo + 1;
        nv = n_local + n_remote;
    }
};

// The pair's merged visit list: the K tiles needed by ANY of its four query tiles.  UMMA "tile i" (i = 0, 1) is M = 256
// across the pair: rows 0-127 are query block qbA + i of CTA 0, rows 128-255 query block qbB + i of CTA 1.  With an even
// GQA group the two CTAs hold two heads on the SAME blocks (qbA = qbB); the lone head of an odd group (and every head
// of MHA) is served by one pair on four consecutive blocks of that head (qbB = qbA + 2).  A tile takes part in a visit
// when either CTA's block needs the key tile; the block that does not need it sees the visit fully masked (the masks in
// the softmax are the exact per-row rule, whatever the tile), so no special case exists below this struct.
struct MPlan {
    int lo0, top0, hi0, rlo0, lo1, top1, hi1, rlo1;   // tile i: local key tiles [lo_i, top_i], remote [rlo_i, hi_i] (joint over the CTAs)
    int lo_m, top_m, hi_m, rlo_m, n_loc, n_rem, nm;
    bool bifocal;
    __device__ MPlan(int qbA, int qbB, int n_qb, long long w0, bool bifocal_, int window_only) : bifocal(bifocal_) {
        lo0 = lo1 = rlo0 = rlo1 = 1 << 30; top0 = top1 = -1; hi0 = hi1 = -1;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int qb = (c ? qbB : qbA) + i;
                if (qb >= n_qb) continue;
                const Plan t(qb, w0, bifocal, window_only);
                int& lo = i ? lo1 : lo0; int& top = i ? top1 : top0; int& hi = i ? hi1 : hi0; int& rlo = i ? rlo1 : rlo0;
                if (t.n_local > 0) { lo = t.kt_lo < lo ? t.kt_lo : lo; top = qb > top ? qb : top; }
                if (t.n_remote > 0) { hi = t.kt_hi > hi ? t.kt_hi : hi; rlo = t.kt_rlo < rlo ? t.kt_rlo : rlo; }
            }
        }
        lo_m = lo0 < lo1 ? lo0 : lo1;
        top_m = top0 > top1 ? top0 : top1;
        hi_m = hi0 > hi1 ? hi0 : hi1;
        rlo_m = rlo0 < rlo1 ? rlo0 : rlo1;
        n_loc = top_m >= lo_m ? top_m - lo_m + 1 : 0;
        n_rem = hi_m >= rlo_m ? hi_m - rlo_m + 1 : 0;
        nm = n_loc + n_rem;
    }
    __device__ __forceinline__ Visit at(int m) const {
        Visit x;
        if (m < n_loc) { x.kt = top_m - m; x.mode = bifocal ? 1 : 0; }
        else { x.kt = hi_m - (m - n_loc); x.mode = 2; }
        return x;
    }
    __device__ __forceinline__ bool part(int i, const Visit& x) const {
        const int lo = i ? lo1 : lo0, top = i ? top1 : top0, hi = i ? hi1 : hi0, rlo = i ? rlo1 : rlo0;
        return x.mode == 2 ? (x.kt <= hi && x.kt >= rlo) : (x.kt >= lo && x.kt <= top);
    }
};

// Softmax exponentials of one row, 32 columns per block, software-pipelined by hand: ptxas puts the FADD2 / F2FP that
// consume an exponential directly behind its MUFU.EX2, and the in-order warp then stalls one MUFU latency per pair
// (measured: 1.7-1.9 k cycles for 128 columns).  Here a block's scores first become exp2 arguments (exp_args), then its
// exponentials are issued while the sums and bf16 packs of the PREVIOUS block are interleaved (exp_issue_consume).
__device__ __forceinline__ void exp_args(uint32_t (&sx)[32], uint64_t sl2x2, uint64_t mneg2) {
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
        const uint64_t xx = ffma2(pack2(__uint_as_float(sx[j]), __uint_as_float(sx[j + 1])), sl2x2, mneg2);
        float x0, x1;
        unpack2(xx, x0, x1);
        sx[j] = __float_as_uint(x0); sx[j + 1] = __float_as_uint(x1);
    }
}
__device__ __forceinline__ float ex2v(float x) {                      // volatile: keeps the issue order written here
    float y;
    asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// volatile as well: ptxas otherwise hoists these consumers back up to their MUFU.EX2
__device__ __forceinline__ uint64_t fadd2v(uint64_t a, uint64_t b) {
    uint64_t y;
    asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(y) : "l"(a), "l"(b));
    return y;
}
__device__ __forceinline__ uint32_t bf16x2v(float lo, float hi) {
    uint32_t y;
    asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(y) : "f"(hi), "f"(lo));
    return y;
}
__device__ __forceinline__ void consume_pair(const uint32_t (&pp)[32], int j, uint64_t& l2a, uint64_t& l2b, uint32_t (&pk)[16]) {
    const float p0 = __uint_as_float(pp[j]), p1 = __uint_as_float(pp[j + 1]);
    if (j & 2) l2b = fadd2v(l2b, pack2(p0, p1)); else l2a = fadd2v(l2a, pack2(p0, p1));
    pk[j >> 1] = bf16x2v(p0, p1);
}
// exponentials of block `cur` (in place); the row sums and P words of block `prev` (already exponentiated) in between
template <bool HAS_PREV>
__device__ __forceinline__ void exp_issue_consume(uint32_t (&cur)[32], const uint32_t (&prev)[32], uint64_t& l2a, uint64_t& l2b,
                                                  uint32_t (&pk)[16]) {
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
        if ((j & 6) < 2 * POLY_OF_4) {                                 // this pair on the FMA pipe (scores here are finite)
            float r0, r1;
            exp2_poly2(pack2(__uint_as_float(cur[j]), __uint_as_float(cur[j + 1])), r0, r1);
            cur[j] = __float_as_uint(r0); cur[j + 1] = __float_as_uint(r1);
        } else {
            cur[j] = __float_as_uint(ex2v(__uint_as_float(cur[j])));
            cur[j + 1] = __float_as_uint(ex2v(__uint_as_float(cur[j + 1])));
        }
        if (HAS_PREV) consume_pair(prev, j, l2a, l2b, pk);
    }
}
__device__ __forceinline__ void consume_block(const uint32_t (&pp)[32], uint64_t& l2a, uint64_t& l2b, uint32_t (&pk)[16]) {
#pragma unroll
    for (int j = 0; j < 32; j += 2) consume_pair(pp, j, l2a, l2b, pk);
}

__device__ __forceinline__ float max32(const uint32_t (&s)[32], float m) {
    float a = m, b = -INFINITY, c = -INFINITY, d = -INFINITY;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        a = max3(a, __uint_as_float(s[j]), __uint_as_float(s[j + 1]));
        b = max3(b, __uint_as_float(s[j + 2]), __uint_as_float(s[j + 3]));
        c = max3(c, __uint_as_float(s[j + 4]), __uint_as_float(s[j + 5]));
        d = max3(d, __uint_as_float(s[j + 6]), __uint_as_float(s[j + 7]));
    }
    return fmaxf(fmaxf(a, b), fmaxf(c, d));
}

__device__ __forceinline__ void mask32(uint32_t (&s)[32], int lo, int hi) {   // keep columns lo..hi of this 32-column block
#pragma unroll
    for (int j = 0; j < 32; ++j)
        if (j < lo || j > hi) s[j] = 0xff800000u;                      // -inf: exp2 -> 0, never wins the max
}

constexpr uint32_t IDESC_QK_BF16 = idesc_f16(1, 1, 0, 0, 2 * BM, BN);
constexpr uint32_t IDESC_QK_F16 = idesc_f16(0, 0, 0, 0, 2 * BM, BN);
constexpr uint32_t IDESC_QK_E5M2 = idesc_f16(1, 1, 0, 0, 2 * BM, BN);   // kind::f8f6f4: format code 1 = e5m2
constexpr uint32_t IDESC_PV = idesc_f16(1, 1, 0, 1, 2 * BM, D);         // A = P (TMEM, bf16), B = V (smem, MN-major)
// the lean rotation (rot.cuh: rotate_rows2) stores -lo; the negate-A / negate-B bits of the descriptor undo the sign
constexpr uint32_t IDESC_NEG_A = 1u << 13, IDESC_NEG_B = 1u << 14;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
prefill_umma2_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                     const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmKh,
                     const __grid_constant__ CUtensorMap tmKe, const __grid_constant__ CUtensorMap tmKl, const Params p) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int cta = (int)cluster_ctarank();
    const int unit = (int)(blockIdx.x >> 1);
    // work units, heaviest query blocks first.  Even GQA group: a unit = (256-row block sb, head pair).  Odd group (g = 2 pp + 1,
    // MHA included): per 512-row block s4 and KV head, pp head pairs on each of its two 256-row blocks and one LONE-head
    // unit that covers all four 128-row blocks of the last head of the group (CTA c takes blocks 4 s4 + 2 c, + 1).
    int head, kvh, qbA, qbB;
    if ((p.g & 1) == 0) {
        const int pairs = p.H_q / 2;
        const int sb = p.n_sb - 1 - unit / pairs;
        const int h0 = 2 * (unit % pairs);
        head = h0 + cta; kvh = h0 / p.g; qbA = qbB = 2 * sb;
    } else {
        const int pp = p.g / 2, npair = p.H_kv * pp;
        const int s4 = p.n_s4 - 1 - unit / p.H_q, j = unit % p.H_q;
        if (j < 2 * npair) {
            const int pi = j < npair ? j : j - npair;
            kvh = pi / pp; head = kvh * p.g + 2 * (pi % pp) + cta;
            qbA = qbB = 2 * (2 * s4 + (j < npair ? 1 : 0));
        } else {
            kvh = j - 2 * npair; head = kvh * p.g + p.g - 1;
            qbA = 4 * s4; qbB = 4 * s4 + 2;
        }
    }
    const int qb0 = cta ? qbB : qbA;                               // this CTA's first query block
    const bool bifocal = p.bifocal != 0;
    const MPlan mp(qbA, qbB, p.n_qb, p.w0, bifocal, p.window_only);
    // 0 fast, 2 e5m2 cross terms, 3 e5m2 cross terms over the two highest-energy pairs of every 8-pair chunk; a KV head
    // whose other channels are too loud falls back from 3 to 2
    int precise = (bifocal && mp.n_rem > 0) ? p.precise : 0;
    if (precise == 3 && __ldg(p.selinfo + kvh * 16 + 8) != 0u) precise = 2;
    // 4: the selected pairs' cross terms in fp16 instead of e5m2 -- asked for, or flagged by the selection kernel when a selected
    // pair is loud in Q and in K at once; the workspace variant's scratch has no fp16 form of the compact rows
    else if (precise == 3 && !p.prerot && __ldg(p.selinfo + kvh * 16 + 9) != 0u) precise = 4;
    if (precise == 4 && p.prerot) precise = 3;
    // shared memory: Q tiles | cross-term Q' operands | K ring | V ring | barriers
    const int QX_BYTES = precise == 3 ? QBOX : precise == 4 ? 2 * QBOX : precise == 2 ? 4 * QBOX : 0;
    const int KST = KH_BYTES + ((precise == 3 || precise == 4) ? KBOX : precise == 2 ? 2 * KBOX : 0);
    const int NK = (precise == 3 || precise == 4) ? 4 : precise == 2 ? 2 : 5;
    const int NV = precise == 3 ? 3 : (precise == 2 || precise == 4) ? 2 : 5;
    unsigned char* sQ = smem;
    unsigned char* sQX = smem + Q_BYTES;
    unsigned char* kring = sQX + QX_BYTES;
    unsigned char* vring = kring + NK * KST;
    Bars* bars = reinterpret_cast<Bars*>(smem + Q_BYTES + RING_BYTES);
    auto sK = [&](int st) { return kring + st * KST; };
    auto sKl = [&](int st) { return kring + st * KST + KH_BYTES; };
    auto sV = [&](int st) { return vring + st * VH_BYTES; };

    if (tid == 0) {
        for (int i = 0; i < NKMAX; ++i) { mbar_init(&bars->k_full[i], 1); mbar_init(&bars->k_ready[i], 8); mbar_init(&bars->k_empty[i], 1); }
        for (int i = 0; i < NVMAX; ++i) { mbar_init(&bars->v_full[i], 1); mbar_init(&bars->v_ready[i], 1); mbar_init(&bars->v_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&bars->s_full[i], 1); mbar_init(&bars->p_full[i], 8); mbar_init(&bars->p_half[i], 8); mbar_init(&bars->pv_done[i], 1); }
        mbar_init(&bars->o_full, 1); mbar_init(&bars->q_full, 1); mbar_init(&bars->q_ready, 8);
        mbar_init(&bars->q_local_done, 1); mbar_init(&bars->q_rot_done, 8);
        fence_barrier_init();
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV);
        if (p.prerot) { prefetch_tmap(&tmKh); prefetch_tmap(&tmKe); prefetch_tmap(&tmKl); }
    }
    if (warp == W_MMA) tmem_alloc2<512>(&bars->tmem_base);
    tc_fence_before();
    cluster_sync_all();                                            // barriers of both CTAs initialised, TMEM allocated
    tc_fence_after();
    const uint32_t tmem = bars->tmem_base;

    if (warp >= 12) {
        reg_dec<REGS_MISC>();
        if (warp == W_KLOAD) {
            // ===================== Q and K producer (each CTA loads its head's Q tiles and its 64 keys of every K tile) =====
            if (lane == 0) {
                mbar_arrive_expect_tx(&bars->q_full, Q_BYTES);      // rows beyond L (a missing second tile) arrive as zeros
                for (int i = 0; i < 2; ++i) {
                    tma_load_3d(sQ + i * QT_BYTES, &tmQ, &bars->q_full, 0, head, (qb0 + i) * BM);
                    tma_load_3d(sQ + i * QT_BYTES + QBOX, &tmQ, &bars->q_full, 64, head, (qb0 + i) * BM);
                }
                Ring rk(NK);
                for (int m = 0; m < mp.nm; ++m, rk.next()) {
                    const Visit x = mp.at(m);
                    const int st = rk.s;
                    TR(4, m, 0);
                    if (m >= NK) mbar_wait_sleep(&bars->k_empty[st], rk.ph ^ 1u);
                    TR(4, m, 1);
                    if (p.prerot && x.mode == 2) {
                        // workspace variant: K' hi (fp16) and the e5m2 cross-term operands come from the scratch
                        mbar_arrive_expect_tx(&bars->k_full[st], KH_BYTES + (precise == 2 ? 2 * KBOX : precise == 3 ? KBOX : 0));
                        tma_load_3d(sK(st), &tmKh, &bars->k_full[st], 0, kvh, x.kt * BN + 64 * cta);
                        tma_load_3d(sK(st) + KBOX, &tmKh, &bars->k_full[st], 64, kvh, x.kt * BN + 64 * cta);
                        if (precise >= 2) tma_load_3d(sKl(st), &tmKe, &bars->k_full[st], 0, kvh, x.kt * BN + 64 * cta);
                        if (precise == 2) tma_load_3d(sKl(st) + KBOX, &tmKl, &bars->k_full[st], 0, kvh, x.kt * BN + 64 * cta);
                    } else {
                        mbar_arrive_expect_tx(&bars->k_full[st], KH_BYTES);
                        tma_load_3d(sK(st), &tmK, &bars->k_full[st], 0, kvh, x.kt * BN + 64 * cta);
                        tma_load_3d(sK(st) + KBOX, &tmK, &bars->k_full[st], 64, kvh, x.kt * BN + 64 * cta);
                    }
                }
            }
        } else if (warp == W_VLOAD) {
            // ===================== V producer (each CTA loads its 64 channels of the tile) =====================
            if (lane == 0) {
                Ring rv(NV);
                for (int m = 0; m < mp.nm; ++m, rv.next()) {
                    const Visit x = mp.at(m);
                    if (m >= NV) mbar_wait_sleep(&bars->v_empty[rv.s], rv.ph ^ 1u);
                    mbar_arrive_expect_tx(&bars->v_full[rv.s], VH_BYTES);
                    tma_load_3d(sV(rv.s), &tmV, &bars->v_full[rv.s], 64 * cta, kvh, x.kt * BN);
                }
            }
        } else if (warp == W_MMA && cta == 1) {
            // ===================== non-leader CTA: tell the leader when our V half has landed =====================
            if (lane == 0) {
                Ring rv(NV);
                for (int m = 0; m < mp.nm; ++m, rv.next()) {
                    mbar_wait_sleep(&bars->v_full[rv.s], rv.ph);
                    mbar_arrive_leader(&bars->v_ready[rv.s]);
                }
            }
        } else if (warp == W_MMA) {
            // ===================== MMA issuer (leader CTA; the warp runs convergently, one elected lane issues) ===========
            const uint32_t tm = __shfl_sync(0xffffffffu, tmem, 0);
            const uint32_t q0a = __shfl_sync(0xffffffffu, smem_u32(sQ), 0);
            const uint32_t qxa = __shfl_sync(0xffffffffu, smem_u32(sQX), 0);
            const uint32_t kring0 = __shfl_sync(0xffffffffu, smem_u32(kring), 0);
            const uint32_t vring0 = __shfl_sync(0xffffffffu, smem_u32(vring), 0);
            Ring rk(NK), rv(NV);
            const uint32_t el = elect_one() ? 1u : 0u;               // the issuing lane; every lane runs the uniform arithmetic
            const uint32_t HI_K = desc_hi_sw128(1024), HI_V = desc_hi_sw128(1024);
            const uint32_t q_lo0 = desc_lo(q0a, 16), qx_lo0 = desc_lo(qxa, 16);
            const uint32_t k_lo0 = desc_lo(kring0, 16), v_lo0 = desc_lo(vring0, VH_BYTES);
            // S_i = Q_i K^T of one visit (K stage kst), then the arrival for the tile's softmax group
            auto qk = [&](int i, int mode, int kst) {
                const uint32_t dS = tm + TM_S + i * 128;
                const uint32_t qa = q_lo0 + (uint32_t)(i * (QT_BYTES >> 4));
                const uint32_t kb = k_lo0 + (uint32_t)((kst * KST) >> 4), klb = kb + (KH_BYTES >> 4);
                const uint32_t idesc = (mode == 2 || p.qk_f16) ? IDESC_QK_F16 : IDESC_QK_BF16;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks)
                    umma2_ss_e(dS, qa + (((ks >> 2) * QBOX + (ks & 3) * 32) >> 4), HI_K,
                               kb + (((ks >> 2) * KBOX + (ks & 3) * 32) >> 4), HI_K, idesc, ks > 0 ? 1u : 0u, el);
                // cross terms: Q' lo (written by this kernel) is stored negated; so is K' lo unless it comes from the workspace
                const uint32_t id_hl = IDESC_QK_E5M2 | (p.prerot ? 0u : IDESC_NEG_B), id_lh = IDESC_QK_E5M2 | IDESC_NEG_A;
                if (mode == 2 && precise == 3) {
                    // compact operands: Q' row = [HI | LO] regions of 32 bytes (tile i at byte 64 i), K' row = [LO | HI]
                    umma2_ss_f8_e(dS, qx_lo0 + 4 * i, HI_K, klb, HI_K, id_hl, 1u, el);
                    umma2_ss_f8_e(dS, qx_lo0 + 4 * i + 2, HI_K, klb + 2, HI_K, id_lh, 1u, el);
                } else if (mode == 2 && precise == 4) {
                    // fp16 compact operands: Q' row of tile i (its own box) = [HI | LO] regions of 64 bytes, K' row = [LO | HI]
                    const uint32_t q4 = qx_lo0 + (uint32_t)((i * QBOX) >> 4);
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks)
                        umma2_ss_e(dS, q4 + 2 * ks, HI_K, klb + 2 * ks, HI_K, IDESC_QK_F16 | IDESC_NEG_B, 1u, el);
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks)
                        umma2_ss_e(dS, q4 + 4 + 2 * ks, HI_K, klb + 4 + 2 * ks, HI_K, IDESC_QK_F16 | IDESC_NEG_A, 1u, el);
                } else if (mode == 2 && precise == 2) {
                    const uint32_t qe = qx_lo0 + (uint32_t)(i * ((2 * QBOX) >> 4));   // [Q' e5m2 | Q' lo e5m2] of tile i
#pragma unroll
                    for (int ks = 0; ks < D / 32; ++ks)              // Q' (e5m2) . K' lo (e5m2)
                        umma2_ss_f8_e(dS, qe + 2 * ks, HI_K, klb + (KBOX >> 4) + 2 * ks, HI_K, id_hl, 1u, el);
#pragma unroll
                    for (int ks = 0; ks < D / 32; ++ks)              // Q' lo (e5m2) . K' (e5m2)
                        umma2_ss_f8_e(dS, qe + (QBOX >> 4) + 2 * ks, HI_K, klb + 2 * ks, HI_K, id_lh, 1u, el);
                }
                umma2_commit_e(&bars->s_full[i], el);
            };
            // the K stage of visit m is free once its Q K^T (of both tiles) have completed
            auto qk_finish = [&](int m) {
                umma2_commit_e(&bars->k_empty[rk.s], el);
                if (mp.n_rem > 0 && m == mp.n_loc - 1) umma2_commit_e(&bars->q_local_done, el);
                rk.next();
            };
            // O_i += P_i V over keys [64 half, 64 half + 64) of the tile
            auto pv = [&](int i, int vst, bool first, int half) {
                const uint32_t vb = v_lo0 + (uint32_t)((vst * VH_BYTES) >> 4);
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                    const int ks = 4 * half + k4;
                    umma2_ts_e(tm + TM_O + i * 128, tm + TM_S + i * 128 + ks * 8, vb + ((ks * 2048) >> 4), HI_V, IDESC_PV,
                               (!first || ks > 0) ? 1u : 0u, el);
                }
                if (half) umma2_commit_e(&bars->pv_done[i], el);
            };
            mbar_wait_sleep(&bars->q_ready, 0);
            uint32_t jp = 0, started = 0;                            // per tile (bit i): parity of the next P V, any P V issued
            // step m issues P_i V of visit m and Q_i K^T of visit m + 1, tile by tile (m = -1: only the first Q K^T).  When
            // visit m + 1 is the first remote one, the P V go first and the Q K^T wait for Q' (second pass).
            for (int m = -1; m < mp.nm; ++m) {
                const bool has_pv = m >= 0, has_next = m + 1 < mp.nm;
                const Visit x = mp.at(has_pv ? m : 0);
                const Visit y = mp.at(has_next ? m + 1 : 0);
                const bool sw = has_next && y.mode == 2 && m + 1 == mp.n_loc;
                if (has_pv) {
                    TR(0, m, 6);
                    mbar_wait_sleep(&bars->v_full[rv.s], rv.ph);           // our V half ...
                    mbar_wait_sleep(&bars->v_ready[rv.s], rv.ph);          // ... and the other CTA's
                    TR(0, m, 7);
                }
                bool kw = false;
#pragma unroll 1
                for (int pass = 0; pass < (sw ? 2 : 1); ++pass) {
                    if (pass == 1) mbar_wait_sleep(&bars->q_rot_done, 0);
#pragma unroll 1
                    for (int i = 0; i < 2; ++i) {
                        if (pass == 0 && has_pv && mp.part(i, x)) {
                            TR(0, m, 2 * i);
                            mbar_wait_sleep(&bars->p_half[i], (jp >> i) & 1u);
                            tc_fence_after();
                            pv(i, rv.s, !((started >> i) & 1u), 0);
                            mbar_wait_sleep(&bars->p_full[i], (jp >> i) & 1u);
                            TR(0, m, 2 * i + 1);
                            tc_fence_after();
                            pv(i, rv.s, !((started >> i) & 1u), 1);
                            jp ^= 1u << i;
                            started |= 1u << i;
                        }
                        if (pass == (sw ? 1 : 0) && has_next && mp.part(i, y)) {
                            if (!kw) { TR(0, m, 4); mbar_wait_sleep(&bars->k_ready[rk.s], rk.ph); TR(0, m, 5); tc_fence_after(); kw = true; }
                            qk(i, y.mode, rk.s);
                        }
                    }
                }
                if (has_pv) {
                    umma2_commit_e(&bars->v_empty[rv.s], el);
                    rv.next();
                }
                if (has_next) qk_finish(m + 1);
            }
            umma2_commit_e(&bars->o_full, el);
        }
    } else if (warp < 4) {
        // ===================== rotate group (steps a4, a5) =====================
        reg_dec<REGS_ROT>();
        mbar_wait_sleep(&bars->q_full, 0);
        if (lane == 0) mbar_arrive_leader(&bars->q_ready);
        const bool rotating = mp.n_rem > 0 && !p.prerot;
        const uint32_t selw = (mp.n_rem > 0 && p.selinfo) ? __ldg(p.selinfo + kvh * 16 + (tid & 7)) : 0u;
        // one visit loop per operand mode, chosen once per CTA, so the hot loop carries no mode switches (code size)
        auto visit_loop = [&](auto mode_tag) {
            constexpr int KM = decltype(mode_tag)::value;             // 0 hi only, 2 full e5m2 copies, 5 compact selective rows
            KRot<4> rot;
            SelTree sel;
            sel.init(selw);
            if (mp.n_rem > 0) {
                rot.init(p.lo, p.hi, tid, p.G, 0);
                if (rotating) rot.prefetch((unsigned)(mp.hi_m * BN + 64 * cta));     // first remote visit
            }
            Ring rk(NK);
#pragma unroll 1
            for (int m = 0; m < mp.nm; ++m, rk.next()) {
                const Visit x = mp.at(m);
                const int st = rk.s;
                TR(3, m, 0);
                mbar_wait_sleep(&bars->k_full[st], rk.ph);
                TR(3, m, 1);
                if (x.mode == 2) {
                    if (rotating) {
                        rotate_rows2<4, KBOX, KM>(smem_u32(sK(st)), smem_u32(sKl(st)), (unsigned)(x.kt * BN + 64 * cta), rot, sel, 0u, KM == 6 ? 64u : 32u);
                        fence_proxy_async_smem();
                        if (x.kt > 0) rot.prefetch((unsigned)((x.kt - 1) * BN + 64 * cta));   // next remote visit's first row
                    }
                    if (m == mp.n_loc) {
                        // first remote visit: Q -> Q' = R(Delta q) Q, in place in shared memory (both tiles, 64 rows per pass)
                        if (mp.n_loc > 0) mbar_wait_sleep(&bars->q_local_done, 0);
#pragma unroll 1
                        for (int pass = 0; pass < 4; ++pass) {
                            const int i = pass >> 1, half = pass & 1;
                            KRot<4> qr;
                            qr.init(p.lo, p.hi, tid, p.G, 64 * half);
                            qr.prefetch((unsigned)((qb0 + i) * BM));
                            const uint32_t qx = KM == 2 ? smem_u32(sQX) + (uint32_t)(i * 2 * QBOX)
                                              : KM == 6 ? smem_u32(sQX) + (uint32_t)(i * QBOX) : smem_u32(sQX);
                            rotate_rows2<4, QBOX, KM>(smem_u32(sQ + i * QT_BYTES), qx, (unsigned)((qb0 + i) * BM), qr, sel,
                                                      KM == 6 ? 64u : 64u * i + 32u, KM == 6 ? 0u : 64u * i);
                        }
                        fence_proxy_async_smem();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_leader(&bars->q_rot_done);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive_leader(&bars->k_ready[st]);
                TR(3, m, 2);
            }
        };
        if (precise == 3) visit_loop(std::integral_constant<int, 5>{});
        else if (precise == 4) visit_loop(std::integral_constant<int, 6>{});
        else if (precise == 2) visit_loop(std::integral_constant<int, 2>{});
        else visit_loop(std::integral_constant<int, 0>{});
    } else {
        // ===================== softmax groups (steps a6-a8): one thread per query row =====================
        reg_inc<REGS_SOFTMAX>();
        const int i = (warp - W_SOFTMAX) >> 2;                         // query tile of this group
        const int quad = warp & 3;
        const int r = (quad << 5) | lane;
        const int qb = qb0 + i;
        const long long q0 = (long long)qb * BM;
        const uint32_t lane_base = (uint32_t)(quad << 5) << 16;
        const uint32_t tS = tmem + lane_base + TM_S + i * 128;
        const uint32_t tO = tmem + lane_base + TM_O + i * 128;
        const float sl2 = (1.0f / sqrtf((float)D)) * kLog2e;
        const uint64_t sl2x2 = pack2(sl2, sl2);
        float m_ref = -INFINITY;
        uint64_t l2a = 0, l2b = 0;                                     // packed fp32x2 partial row sums
        int v = 0;                                                     // visits this tile has taken part in
        for (int m = 0; m < mp.nm; ++m) {
            const Visit x = mp.at(m);
            if (!mp.part(i, x)) continue;
            const long long k0 = (long long)x.kt * BN;
            const long long qrel = q0 + r - k0;
            int lo = 0, hi = BN - 1;
            bool masked = false;
            if (x.mode != 2 && k0 + BN - 1 > q0) {                                               // causal diagonal
                hi = qrel < hi ? (int)qrel : hi;
                masked = true;
            }
            if (x.mode == 1 && (q0 + BM - 1 - k0 > p.w0)) {                                      // q-k <= w0 (R1)
                const long long a = qrel - p.w0;
                lo = a > 0 ? (int)a : 0;
                masked = true;
            }
            if (x.mode == 2 && p.window_only != 2 && (q0 - (k0 + BN - 1) <= p.w0)) {             // q-k > w0
                const long long a = qrel - p.w0 - 1;
                hi = a < hi ? (int)a : hi;
                masked = true;
            }
            if (x.mode == 2 && p.window_only == 2) {                                             // call C: 0 <= q-k <= w0
                if (k0 + BN - 1 > q0) { hi = qrel < hi ? (int)qrel : hi; masked = true; }
                if (q0 + BM - 1 - k0 > p.w0) { const long long a = qrel - p.w0; lo = a > 0 ? (int)a : 0; masked = true; }
            }
            TR(1 + i, v, 0);
            mbar_wait_sleep(&bars->s_full[i], (uint32_t)v & 1u);
            TR(1 + i, v, 1);
            tc_fence_after();
            uint32_t s0[32], s1[32], s2[32], s3[32];
            tmem_ld32(tS, s0);
            tmem_ld32(tS + 32, s1);
            tmem_ld_wait();
            tmem_ld32(tS + 64, s2);                                    // in flight under the maxima of the first half
            tmem_ld32(tS + 96, s3);
            if (masked) { mask32(s0, lo, hi); mask32(s1, lo - 32, hi - 32); }
            const float mxa = fmaxf(max32(s0, -INFINITY), max32(s1, -INFINITY));
            tmem_ld_wait();
            if (masked) { mask32(s2, lo - 64, hi - 64); mask32(s3, lo - 96, hi - 96); }
            const float mx = fmaxf(mxa, fmaxf(max32(s2, -INFINITY), max32(s3, -INFINITY)));
            const float mnew = mx * sl2;
            TR(1 + i, v, 2);
            if (v == 0) {
                m_ref = mnew;
            } else {
                const bool need = mnew > m_ref + 8.0f;                 // lazy rescale: only on a jump of 2^8
                if (__any_sync(0xffffffffu, need)) {
                    mbar_wait_sleep(&bars->pv_done[i], (uint32_t)(v - 1) & 1u);   // O += P V of visit v-1 must have landed
                    tc_fence_after();
                    const float alpha = need ? ex2(m_ref - mnew) : 1.0f;
                    if (need) m_ref = mnew;
                    const uint64_t al2 = pack2(alpha, alpha);
                    l2a = fmul2(l2a, al2); l2b = fmul2(l2b, al2);
                    uint32_t rg[16];
#pragma unroll 1
                    for (int ch = 0; ch < 8; ++ch) {
                        tmem_ld16(tO + ch * 16, rg);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) rg[j] = __float_as_uint(__uint_as_float(rg[j]) * alpha);
                        tmem_st16(tO + ch * 16, rg);
                    }
                }
            }
            // a row whose every key so far is masked has m_ref = -inf: keep exp2 arguments finite (-> p = 0)
            const float mneg = (m_ref == -INFINITY) ? 0.f : -m_ref;
            const uint64_t mneg2 = pack2(mneg, mneg);
            uint32_t pk[16];
            // P (bf16, columns 0..63 of S_i) overwrites S values that are already in registers
            exp_args(s0, sl2x2, mneg2);
            exp_args(s1, sl2x2, mneg2);
            exp_issue_consume<false>(s0, s0, l2a, l2b, pk);
            exp_args(s2, sl2x2, mneg2);
            exp_issue_consume<true>(s1, s0, l2a, l2b, pk); tmem_st16(tS, pk);
            exp_args(s3, sl2x2, mneg2);
            exp_issue_consume<true>(s2, s1, l2a, l2b, pk); tmem_st16(tS + 16, pk);
            tmem_st_wait();                                            // the first 64 columns of P are in TMEM
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(&bars->p_half[i]);
            exp_issue_consume<true>(s3, s2, l2a, l2b, pk); tmem_st16(tS + 32, pk);
            consume_block(s3, l2a, l2b, pk); tmem_st16(tS + 48, pk);
            TR(1 + i, v, 3);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(&bars->p_full[i]);
            TR(1 + i, v, 4);
            ++v;
        }
        // ---- epilogue (step a8) ----
        if (v > 0) {
            float la, lb, lc, ld;
            unpack2(l2a, la, lb); unpack2(l2b, lc, ld);
            const float l = (la + lb) + (lc + ld);
            mbar_wait_sleep(&bars->o_full, 0);
            tc_fence_after();
            const long long q = q0 + r;
            const float inv = 1.0f / l;
            const bool qok = q < p.L;
            __nv_bfloat16* orow = p.out + ((size_t)(qok ? q : 0) * p.H_q + head) * D;
            float* orow32 = reinterpret_cast<float*>(p.out) + ((size_t)(qok ? q : 0) * p.H_q + head) * D;   // out_f32 (unfused baseline)
#pragma unroll 1
            for (int ch = 0; ch < 4; ++ch) {
                uint32_t rg[32];
                tmem_ld32(tO + ch * 32, rg);
                tmem_ld_wait();
                if (qok && p.out_f32) {
#pragma unroll
                    for (int j = 0; j < 32; j += 4)
                        *reinterpret_cast<float4*>(orow32 + ch * 32 + j) =
                            make_float4(__uint_as_float(rg[j]) * inv, __uint_as_float(rg[j + 1]) * inv,
                                        __uint_as_float(rg[j + 2]) * inv, __uint_as_float(rg[j + 3]) * inv);
                } else if (qok) {
#pragma unroll
                    for (int j = 0; j < 32; j += 8) {
                        uint32_t w[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            w[e] = bf16x2(__uint_as_float(rg[j + 2 * e]) * inv, __uint_as_float(rg[j + 2 * e + 1]) * inv);
                        *reinterpret_cast<uint4*>(orow + ch * 32 + j) = make_uint4(w[0], w[1], w[2], w[3]);
                    }
                }
            }
            if (qok) p.lse[(size_t)head * p.L + q] = (m_ref + log2f(l)) * 0.6931471805599453f;
        }
    }
    tc_fence_before();
    cluster_sync_all();                                            // the peer may still be reading our smem / TMEM
    if (warp == W_MMA) tmem_dealloc2<512>(tmem);
}

}  // namespace

#ifdef JL_TRACE
extern "C" int jetlong_debug_trace(long long* dst, int n, int block) {
    const int total = TR_ROLES * TR_M * TR_SLOTS;
    if (dst && cudaMemcpyFromSymbol(dst, g_trace, sizeof(long long) * (n < total ? n : total)) != cudaSuccess) return -1;
    if (cudaMemcpyToSymbol(g_trace_block, &block, sizeof(int)) != cudaSuccess) return -1;
    return total;
}
#endif

int launch_prefill_v2(const PrefillV2Args& a, cudaStream_t st) {
    Params p;
    p.out = (__nv_bfloat16*)a.out; p.lse = a.lse;
    p.L = a.L; p.w0 = a.w0; p.G = a.G;
    p.H_q = a.H_q; p.H_kv = a.H_kv; p.g = a.H_q / a.H_kv;
    p.bifocal = a.bifocal; p.precise = a.precise; p.prerot = a.prerot; p.window_only = a.window_only; p.qk_f16 = a.qk_f16; p.out_f32 = a.out_f32;
    p.n_qb = (int)((a.L + BM - 1) / BM);
    const int qb_hi = (a.qb_hi < 0 || a.qb_hi > p.n_qb) ? p.n_qb : a.qb_hi;
    if ((a.qb_lo & 3) || a.qb_lo < 0 || a.qb_lo >= qb_hi) return JETLONG_INVALID_ARG;
    p.n_sb = (qb_hi + 1) / 2;
    p.n_s4 = (qb_hi + 3) / 4;
    p.lo = a.lo; p.hi = a.hi; p.selinfo = a.selinfo;
    if (cudaFuncSetAttribute(prefill_umma2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess)
        return check_launch("prefill_umma2 attr");
    const unsigned grid = (p.g & 1) ? 2u * (unsigned)(p.n_s4 - a.qb_lo / 4) * (unsigned)a.H_q
                                    : 2u * (unsigned)(p.n_sb - a.qb_lo / 2) * (unsigned)(a.H_q / 2);
    prefill_umma2_kernel<<<grid, NTHREADS, SMEM_BYTES, st>>>(a.tmQ, a.tmK, a.tmV, a.tmKh, a.tmKe, a.tmKl, p);
    note_launch();
    return check_launch("prefill_umma2_kernel");
}

}  // namespace jetlong
