// prefill_umma.cu -- tcgen05 UMMA bifocal / causal prefill for bf16, head_dim 128 (steps a3-a8, a10).
//
// One CTA PAIR (cluster of 2, tcgen05 cta_group::2) = 128 query rows x 2 query heads of one KV group: both
// heads see the same keys, the same positions and therefore the same tile classification.  Every UMMA is
// M = 256 across the pair (CTA c owns head h0 + c), so each CTA stages and -- on remote visits -- rotates only
// HALF of every K tile (its 64 keys) and loads half of every V tile (its 64 channels).
// Warp roles (448 threads per CTA; ptxas caps >384 threads at 128 registers, the kernel uses 124, no spills):
//   warp 0      TMA producer: its half of K and V per visit, SWIZZLE_128B boxes, NS-stage ring
//   warp 1      MMA issuer (leader CTA only, one thread): S_b = Q K^T (A = Q from TMEM), O += P V (A = P from TMEM)
//   warps 2-5   rotate group: stages Q into TMEM; on remote visits rotates its K half in shared memory between
//               the TMA load and the MMA (Eq.(6): bf16 -> fp32 rotate -> fp16 hi (+ fp16 lo)); once per CTA
//               it replaces Q in TMEM by Q' = R(Delta q) Q (hi, lo)
//   warps 6-13  softmax groups: two threads per query row (64 keys of the tile each, S kept in registers, row max
//               combined through shared memory), online softmax over the visits, epilogue
// TMEM (512 columns): S0 | S1 | O | Qa | Qb  (128, 128, 128, 64, 64).  P (bf16) aliases columns 0..63 of its S.
// S is double-buffered over consecutive visits so QK^T of visit v+1 overlaps the softmax of visit v.
//
// Visit order per pair: local visits first (diagonal tile, then the band down to q - w0), then the Q -> Q'
// switch, then the remote visits.  The straddle tile is visited twice with complementary masks (step a6).
// All visits feed ONE running (m, l, O) per row: the additive form of the Eq.(7) merge.
//
// Precision: local visits multiply the stored bf16 Q, K exactly.  Remote
// operands are fp32-rotated and split hi + lo in fp16; S = Q'hi K'hi + Q'hi K'lo + Q'lo K'hi (three UMMA
// groups, "compensated").  The fast mode keeps only Q'hi K'hi (one group) and misses the lse tolerance on
// outlier-channel inputs; it is opt-in (jetlong_set_prefill_precision).
#include <cuda.h>
#include <math.h>
#include <mutex>

#include "common.cuh"
#include "umma.cuh"
#include "rot.cuh"
#include "prefill_v2.cuh"

namespace jetlong {

namespace {

using namespace ptx;
using namespace dev;

constexpr int D = 128, BM = 128, BN = 128;
// Two rings: K stages are released as soon as Q K^T of their visit has completed, V stages after P V -- so the K side
// (TMA load -> rotate -> cluster exchange -> MMA) runs several visits ahead of the softmax (r1: one ring of four K|Klo|V
// stages held every K tile until its P V, the K side had ~2 visits of slack and the MMA warp waited ~1.1 k cycles per
// visit for operands).
constexpr int NV = 4;                                 // V ring depth
constexpr int NKMAX = 8;                              // K ring depth = min(NKMAX, K_RING_BYTES / K stage size)
constexpr int KH_BYTES = 64 * D * 2;                  // this CTA's 64 keys: two 8 KB SWIZZLE_128B boxes (ch 0-63 | 64-127)
constexpr int KBOX = 64 * 128;                        // one K box: 64 rows x 128 B
constexpr int VH_BYTES = BN * 64 * 2;                 // this CTA's 64 channels of 128 keys: one 16 KB box
constexpr int K_RING_BYTES = 9 * KH_BYTES;            // 144 KB: 8 stages of K alone, 6 of K | compact lo rows, 4 of K | K lo
constexpr int NTHREADS = 512;
constexpr float kLog2e = 1.4426950408889634f;
constexpr int POLY_OF_4 = 0;                          // of every 4 exponential pairs, this many use the FMA-pipe polynomial.
// Measured on C2 (same box, back to back): 0 -> 25.5 ms, 1 -> 25.4 ms, 2 -> 27.2 ms (default precision); the kernel runs
// under the power cap (~1.45 GHz), where extra FMA instructions cost more clock than the freed MUFU cycles return.
// warp roles.  The scheduler of an SM sub-partition prefers the highest warp id: the MMA issuer and the producers (few
// instructions, all on the critical path) sit above the softmax warps, the rotate group (which runs visits ahead) below.
constexpr int W_KLOAD = 12, W_VLOAD = 13, W_MMA = 15;   // warps 0-3 rotate, 4-11 softmax
constexpr uint32_t TM_S = 0, TM_O = 256, TM_QA = 384, TM_QB = 448;
constexpr uint32_t TM_QY = 448, TM_QR = 480;         // precision mode 2: Q' and Q' lo as e5m2 (32 columns each) in place of Qb

struct Bars {
    uint64_t k_full[NKMAX];    // local: TMA bytes of this CTA's K half landed
    uint64_t k_ready[NKMAX];   // leader: both rotate groups are done with K stage s (8 warp arrivals)
    uint64_t k_empty[NKMAX];   // both: Q K^T reading K stage s has completed (multicast commit)
    uint64_t v_full[NV];       // local: TMA bytes of this CTA's V half landed
    uint64_t v_ready[NV];      // leader: the other CTA's V half has landed (its forwarding warp)
    uint64_t v_empty[NV];      // both: P V reading V stage s has completed (multicast commit)
    uint64_t s_full[2];        // both: S_b holds Q K^T of a visit
    uint64_t p_full[2];        // leader: both softmax groups wrote P_b and are done reading S_b (8 warp arrivals)
    uint64_t pv_done;          // both: O += P V of a visit has completed
    uint64_t o_full;           // both: all MMAs done
    uint64_t q_ready;          // leader: Q staged in TMEM by both rotate groups
    uint64_t q_local_done;     // both: the last local Q K^T has completed, Qa may be overwritten
    uint64_t q_rot_done;       // leader: Q' (hi, lo) staged in TMEM
    uint32_t tmem_base;
    float xchg[4 * BM];        // row-max / row-sum exchange between the two column halves of a row
};

constexpr size_t SMEM_BYTES = 1024 /*align slack*/ + (size_t)NV * VH_BYTES + K_RING_BYTES + 4096 /*Bars*/;
static_assert(SMEM_BYTES <= 232448, "shared memory budget");
static_assert(sizeof(Bars) <= 4096, "Bars");

// position in a ring of n stages: stage s, phase parity ph of the current use
struct Ring {
    int n, s;
    uint32_t ph;
    __device__ Ring(int n_, int start = 0) : n(n_), s(start % n_), ph((uint32_t)(start / n_) & 1u) {}
    __device__ __forceinline__ void next() { if (++s == n) { s = 0; ph ^= 1u; } }
};

struct Params {
    const __nv_bfloat16* Q;
    __nv_bfloat16* out;
    float* lse;
    long long L, w0, G;
    int H_q, H_kv, g;
    int bifocal, precise;
    int prerot;                                       // remote K tiles come pre-rotated from the workspace (8(f)-1)
    int window_only;                                  // only the local band 0 <= q-k <= w0 (calls A and C of the unfused path)
    int qk_f16;                                       // Q and K hold fp16 (pre-rotated operands of calls B and C), not bf16
    int qb_top, qb_lo;                                // this launch covers query blocks [qb_lo, qb_top), heaviest first
    const float2* lo;
    const float2* hi;
    const uint32_t* selinfo;                          // [H_kv][16]: 8 PRMT selectors (two pairs per 8-pair chunk), full-mode flag
};

struct Visit { int kt; int mode; };                   // mode 0 = causal/control, 1 = local, 2 = remote

struct Plan {
    int qb, n_local, n_remote, kt_hi, nv;
    __device__ Plan(int qb_, long long w0, bool bifocal, bool window_only = false) : qb(qb_) {
        const long long q0 = (long long)qb * BM;
        if (!bifocal) { n_local = qb + 1; n_remote = 0; kt_hi = -1; nv = n_local; return; }
        long long t = q0 - w0 - (BN - 1);                              // local iff k0 >= t
        long long kt_lo = t <= 0 ? 0 : (t + BN - 1) / BN;
        n_local = (int)(qb - kt_lo + 1);
        long long u = q0 + (BM - 1) - 1 - w0;                          // remote iff k0 <= u  (q0+127-k0 > w0)
        kt_hi = u < 0 ? -1 : (int)(u / BN);
        if (kt_hi > qb) kt_hi = qb;
        n_remote = kt_hi + 1;
        if (window_only) { n_remote = 0; kt_hi = -1; }
        nv = n_local + n_remote;
    }
    __device__ Visit at(int v, bool bifocal) const {
        Visit x;
        if (v < n_local) { x.kt = qb - v; x.mode = bifocal ? 1 : 0; }
        else { x.kt = kt_hi - (v - n_local); x.mode = 2; }
        return x;
    }
};

// ---- Q staging (step a4): thread = one query row; TMEM column c of Qa/Qb holds channels (2c, 2c+1) ------------
__device__ __forceinline__ void stage_q_raw(const __nv_bfloat16* qrow, bool valid, uint32_t tQa) {
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        uint4 u = make_uint4(0, 0, 0, 0);
        if (valid) u = __ldg(reinterpret_cast<const uint4*>(qrow) + j);
        tmem_st4(tQa + 4 * j, u.x, u.y, u.z, u.w);
    }
}
__device__ __forceinline__ void stage_q_rot(const __nv_bfloat16* qrow, bool valid, long long q, long long G,
                                            const float2* __restrict__ lo, const float2* __restrict__ hi,
                                            uint32_t tQa, uint32_t tQb, int precise, const uint32_t* __restrict__ sel) {
#pragma unroll 1
    for (int jp = 0; jp < 4; ++jp) {
        uint32_t w[4] = {0u, 0u, 0u, 0u};                    // precise 3: compact hi1 | hi2 | lo1 | lo2 words of chunks 2jp, 2jp+1
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int j = 2 * jp + u;                         // channels 8j..8j+7 and 64+8j..
            uint4 u1 = make_uint4(0, 0, 0, 0), u2 = u1;
            if (valid) {
                u1 = __ldg(reinterpret_cast<const uint4*>(qrow) + j);
                u2 = __ldg(reinterpret_cast<const uint4*>(qrow) + 8 + j);
            }
            float cs_c[8], cs_s[8];
            cs8(lo, hi, q, G, 8 * j, cs_c, cs_s);
            const uint32_t a[4] = {u1.x, u1.y, u1.z, u1.w}, b[4] = {u2.x, u2.y, u2.z, u2.w};
            uint32_t h1[4], h2[4], l1[4], l2[4];
            rot8(a, b, cs_c, cs_s, h1, h2, l1, l2);
            tmem_st4(tQa + 4 * j, h1[0], h1[1], h1[2], h1[3]);
            tmem_st4(tQa + 32 + 4 * j, h2[0], h2[1], h2[2], h2[3]);
            if (precise == 2) {                                   // e5m2 copies: column c of QY / QR holds channels 4c..4c+3
                tmem_st2(tQb + 2 * j, e5m2x4(h1[0], h1[1]), e5m2x4(h1[2], h1[3]));
                tmem_st2(tQb + 16 + 2 * j, e5m2x4(h2[0], h2[1]), e5m2x4(h2[2], h2[3]));
                tmem_st2(tQb + 32 + 2 * j, e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3]));
                tmem_st2(tQb + 48 + 2 * j, e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]));
            } else if (precise == 3) {                            // the two selected pairs of this chunk, as e5m2
                const uint32_t sj = __ldg(sel + j);
                w[0] |= (__byte_perm(e5m2x4(h1[0], h1[1]), e5m2x4(h1[2], h1[3]), sj) & 0xffffu) << (16 * u);
                w[1] |= (__byte_perm(e5m2x4(h2[0], h2[1]), e5m2x4(h2[2], h2[3]), sj) & 0xffffu) << (16 * u);
                w[2] |= (__byte_perm(e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3]), sj) & 0xffffu) << (16 * u);
                w[3] |= (__byte_perm(e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]), sj) & 0xffffu) << (16 * u);
            } else {
                tmem_st4(tQb + 4 * j, l1[0], l1[1], l1[2], l1[3]);
                tmem_st4(tQb + 32 + 4 * j, l2[0], l2[1], l2[2], l2[3]);
            }
        }
        if (precise == 3) {          // QY' = [hi1 | hi2] in columns 0-7 of Qb, QR' = [lo1 | lo2] in columns 8-15
            tmem_st1(tQb + jp, w[0]);
            tmem_st1(tQb + 4 + jp, w[1]);
            tmem_st1(tQb + 8 + jp, w[2]);
            tmem_st1(tQb + 12 + jp, w[3]);
        }
    }
}

// p = exp2(s * sl2 - m) for 32 scores of a row, packed row sums, bf16 P words.  POLY: of every 4 pairs, POLY_OF_4
// use the FMA-pipe polynomial instead of MUFU.EX2 (never on masked tiles, whose -inf entries need MUFU semantics).
template <bool POLY>
__device__ __forceinline__ void exp_block(const uint32_t (&sx)[32], uint64_t sl2x2, uint64_t mneg2, uint64_t& l2a,
                                          uint64_t& l2b, uint32_t (&pk)[16]) {
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
        const uint64_t xx = ffma2(pack2(__uint_as_float(sx[j]), __uint_as_float(sx[j + 1])), sl2x2, mneg2);
        float p0, p1;
        if (POLY && (j & 6) < 2 * POLY_OF_4) {
            exp2_poly2(xx, p0, p1);
        } else {
            float x0, x1;
            unpack2(xx, x0, x1);
            p0 = ex2(x0); p1 = ex2(x1);
        }
        if (j & 2) l2b = fadd2(l2b, pack2(p0, p1)); else l2a = fadd2(l2a, pack2(p0, p1));
        pk[j >> 1] = bf16x2(p0, p1);
    }
}

constexpr uint32_t IDESC_QK_BF16 = idesc_f16(1, 1, 0, 0, 2 * BM, BN);
constexpr uint32_t IDESC_QK_F16 = idesc_f16(0, 0, 0, 0, 2 * BM, BN);
constexpr uint32_t IDESC_QK_E5M2 = idesc_f16(1, 1, 0, 0, 2 * BM, BN);   // kind::f8f6f4: format code 1 = e5m2
constexpr uint32_t IDESC_PV = idesc_f16(1, 1, 0, 1, 2 * BM, D);  // A = P (TMEM, bf16), B = V (smem, MN-major)

// A cluster is one CTA pair (round 1's clusters of four, which shared rotated K tiles through distributed shared memory,
// were superseded by the two-tile kernel of prefill_umma2.cu and removed).
__device__ __forceinline__ void prefill_body(const CUtensorMap& tmK, const CUtensorMap& tmV, const CUtensorMap& tmKh,
                                             const CUtensorMap& tmKe, const CUtensorMap& tmKl, const Params& p) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    unsigned char* kring = smem + NV * VH_BYTES;
    Bars* bars = reinterpret_cast<Bars*>(kring + K_RING_BYTES);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int rank = (int)cluster_ctarank();
    const int cta = rank & 1;                                      // position in the CTA pair (0 = leader)
    const int pairs = p.H_q / 2;
    const int unit = (int)(blockIdx.x >> 1);
    const int qb = p.qb_top - 1 - unit / pairs;                    // heaviest row blocks first
    const int h0 = 2 * (unit % pairs);
    const int head = h0 + cta;
    const int kvh = h0 / p.g;
    const long long q0 = (long long)qb * BM;
    const bool bifocal = p.bifocal != 0;
    // 0 fast, 1 fp16 cross terms, 2 e5m2 cross terms, 3 e5m2 cross terms over the two highest-energy pairs of every
    // 8-pair chunk; a KV head whose other channels are too loud falls back to 2
    int precise = p.precise;
    if (precise == 3 && __ldg(p.selinfo + kvh * 16 + 8) != 0u) precise = 2;
    Plan plan(qb, p.w0, bifocal, p.window_only != 0);
    const uint32_t own_mask = 3u;
    // K stage = K (hi in place) | cross-term operands; the same for every CTA of the cluster (one KV head)
    const int KST = KH_BYTES + ((!bifocal || p.window_only || precise == 0) ? 0 : precise == 3 ? KBOX : 2 * KBOX);
    const int NK = (K_RING_BYTES / KST) < NKMAX ? (K_RING_BYTES / KST) : NKMAX;
    auto sK = [&](int st) { return kring + st * KST; };
    auto sKl = [&](int st) { return kring + st * KST + KH_BYTES; };
    auto sV = [&](int st) { return smem + st * VH_BYTES; };

    if (tid == 0) {
        for (int i = 0; i < NKMAX; ++i) { mbar_init(&bars->k_full[i], 1); mbar_init(&bars->k_ready[i], 8); mbar_init(&bars->k_empty[i], 1); }
        for (int i = 0; i < NV; ++i) { mbar_init(&bars->v_full[i], 1); mbar_init(&bars->v_ready[i], 1); mbar_init(&bars->v_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&bars->s_full[i], 1); mbar_init(&bars->p_full[i], 16); }
        mbar_init(&bars->pv_done, 1); mbar_init(&bars->o_full, 1); mbar_init(&bars->q_ready, 8);
        mbar_init(&bars->q_local_done, 1); mbar_init(&bars->q_rot_done, 8);
        fence_barrier_init();
        prefetch_tmap(&tmK); prefetch_tmap(&tmV);
        if (p.prerot) { prefetch_tmap(&tmKh); prefetch_tmap(&tmKe); prefetch_tmap(&tmKl); }
    }
    if (warp == W_MMA) tmem_alloc2<512>(&bars->tmem_base);
    tc_fence_before();
    cluster_sync_all();                                            // barriers of both CTAs initialised, TMEM allocated
    tc_fence_after();
    const uint32_t tmem = bars->tmem_base;
    float* xchg = bars->xchg;
    // arrive on the pair leader's copy of a barrier (the leader is rank & ~1 of the cluster)
    auto arrive_leader = [&](uint64_t* bar) {
        mbar_arrive_leader(bar);
    };
    if (warp == W_KLOAD) {
        // ===================== K producer (each CTA loads its 64 keys) =====================
        if (lane == 0) {
            Ring rk(NK);
            for (int v = 0; v < plan.nv; ++v, rk.next()) {
                const Visit x = plan.at(v, bifocal);
                const int st = rk.s;
                if (v >= NK) mbar_wait(&bars->k_empty[st], rk.ph ^ 1u);
                if (p.prerot && x.mode == 2) {
                    // pre-rotated variant: K' hi (fp16) and the e5m2 copies of K' and K' lo come from the workspace
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
            for (int v = 0; v < plan.nv; ++v, rv.next()) {
                const Visit x = plan.at(v, bifocal);
                if (v >= NV) mbar_wait(&bars->v_empty[rv.s], rv.ph ^ 1u);
                mbar_arrive_expect_tx(&bars->v_full[rv.s], VH_BYTES);
                tma_load_3d(sV(rv.s), &tmV, &bars->v_full[rv.s], 64 * cta, kvh, x.kt * BN);
            }
        }
    } else if (warp == W_MMA) {
        if (cta == 1) {
            // ===================== non-leader CTA: tell the leader when our V half has landed =====================
            if (lane == 0) {
                Ring rv(NV);
                for (int v = 0; v < plan.nv; ++v, rv.next()) {
                    mbar_wait(&bars->v_full[rv.s], rv.ph);
                    arrive_leader(&bars->v_ready[rv.s]);
                }
            }
        } else {
        // ===================== MMA issuer (warp 1 of the leader CTA; one elected lane issues) =====================
        // The whole warp runs the loop convergently so that descriptors and TMEM addresses stay in uniform
        // registers; a divergent single-lane issuer costs ~100 cycles of R2UR/ELECT waterfall per MMA (measured).
            const uint32_t tm = __shfl_sync(0xffffffffu, tmem, 0);
            const uint32_t kring0 = __shfl_sync(0xffffffffu, smem_u32(kring), 0);
            const uint32_t vring0 = __shfl_sync(0xffffffffu, smem_u32(smem), 0);
            Ring rq(NK), rvp(NV);                                    // K stage of the next Q K^T, V stage of the next P V
            auto issue_qk = [&](int v) {
                const Visit x = plan.at(v, bifocal);
                const uint32_t dS = tm + TM_S + (v & 1) * 128;
                const uint32_t kb = kring0 + (uint32_t)(rq.s * KST), klb = kb + KH_BYTES;
                if (elect_one()) {
                    if (x.mode != 2) {
                        const uint32_t idesc = p.qk_f16 ? IDESC_QK_F16 : IDESC_QK_BF16;
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks)
                            umma2_ts(dS, tm + TM_QA + ks * 8,
                                     smem_desc_sw128(kb + (ks >> 2) * KBOX + (ks & 3) * 32, 16, 1024), idesc, ks > 0);
                    } else {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks)
                            umma2_ts(dS, tm + TM_QA + ks * 8,
                                     smem_desc_sw128(kb + (ks >> 2) * KBOX + (ks & 3) * 32, 16, 1024), IDESC_QK_F16, ks > 0);
                        if (precise == 2) {
#pragma unroll
                            for (int ks = 0; ks < D / 32; ++ks)      // Q' (e5m2) . K' lo (e5m2)
                                umma2_ts_f8(dS, tm + TM_QY + ks * 8, smem_desc_sw128(klb + KBOX + ks * 32, 16, 1024),
                                            IDESC_QK_E5M2, 1);
#pragma unroll
                            for (int ks = 0; ks < D / 32; ++ks)      // Q' lo (e5m2) . K' (e5m2)
                                umma2_ts_f8(dS, tm + TM_QR + ks * 8, smem_desc_sw128(klb + ks * 32, 16, 1024),
                                            IDESC_QK_E5M2, 1);
                        } else if (precise == 3) {
                            // compact operands: K row = [lo1 | lo2 | hi1 | hi2] (16 B each), Q' = [hi1 | hi2], [lo1 | lo2]
                            umma2_ts_f8(dS, tm + TM_QY, smem_desc_sw128(klb, 16, 1024), IDESC_QK_E5M2, 1);
                            umma2_ts_f8(dS, tm + TM_QY + 8, smem_desc_sw128(klb + 32, 16, 1024), IDESC_QK_E5M2, 1);
                        } else if (precise == 1) {
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks)
                                umma2_ts(dS, tm + TM_QA + ks * 8,
                                         smem_desc_sw128(klb + (ks >> 2) * KBOX + (ks & 3) * 32, 16, 1024), IDESC_QK_F16, 1);
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks)
                                umma2_ts(dS, tm + TM_QB + ks * 8,
                                         smem_desc_sw128(kb + (ks >> 2) * KBOX + (ks & 3) * 32, 16, 1024), IDESC_QK_F16, 1);
                        }
                    }
                    umma2_commit_mask(&bars->s_full[v & 1], own_mask);
                    umma2_commit_mask(&bars->k_empty[rq.s], own_mask);   // the K stage is free again
                    if (plan.n_remote > 0 && v == plan.n_local - 1) umma2_commit_mask(&bars->q_local_done, own_mask);
                }
                __syncwarp();
                rq.next();
            };
            auto issue_pv = [&](int v) {
                mbar_wait(&bars->v_full[rvp.s], rvp.ph);             // our V half ...
                mbar_wait(&bars->v_ready[rvp.s], rvp.ph);            // ... and the other CTA's
                const uint32_t vb = vring0 + (uint32_t)(rvp.s * VH_BYTES);
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < BN / 16; ++ks)
                        umma2_ts(tm + TM_O, tm + TM_S + (v & 1) * 128 + ks * 8,
                                 smem_desc_sw128(vb + ks * 2048, VH_BYTES, 1024), IDESC_PV, (v > 0 || ks > 0) ? 1u : 0u);
                    umma2_commit_mask(&bars->v_empty[rvp.s], own_mask);
                    umma2_commit_mask(&bars->pv_done, own_mask);
                }
                __syncwarp();
                rvp.next();
            };
            auto wait_ready = [&](int) { mbar_wait(&bars->k_ready[rq.s], rq.ph); };   // both rotate groups are done with the stage
            __syncwarp();
            mbar_wait(&bars->q_ready, 0);
            if (plan.nv > 0) {
                if (plan.n_local == 0) mbar_wait(&bars->q_rot_done, 0);
                wait_ready(0);
                tc_fence_after();
                issue_qk(0);
            }
            for (int v = 0; v < plan.nv; ++v) {
                if (v + 1 < plan.nv) {
                    if (plan.n_remote > 0 && v + 1 == plan.n_local) mbar_wait(&bars->q_rot_done, 0);
                    wait_ready(v + 1);
                    tc_fence_after();
                    issue_qk(v + 1);
                }
                mbar_wait(&bars->p_full[v & 1], (v >> 1) & 1);
                tc_fence_after();
                issue_pv(v);
            }
            if (elect_one()) umma2_commit_mask(&bars->o_full, own_mask);
            __syncwarp();
        }
    } else if (warp < 4) {
        // ===================== rotate group (steps a4, a5) =====================
        const int t = tid;                                            // work index for the K rotation
        const uint32_t lane_base = (uint32_t)((warp & 3) << 5) << 16; // TMEM lanes a warp may touch: 32 (warp % 4) ..
        const long long q = q0 + (((warp & 3) << 5) | lane);
        const bool valid = q >= 0 && q < p.L;
        const __nv_bfloat16* qrow = p.Q + ((size_t)(valid ? q : 0) * p.H_q + head) * D;
        stage_q_raw(qrow, valid, tmem + lane_base + TM_QA);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) arrive_leader(&bars->q_ready);
        constexpr int RR = 4;                                         // key rows per rotate thread
        KRot<RR> rot;
        if (plan.n_remote > 0 && !p.prerot) {
            rot.init(p.lo, p.hi, t, p.G, 0);
            rot.prefetch((unsigned)(plan.kt_hi * BN + 64 * cta));     // first remote visit
        }
        Ring rk(NK);
        for (int v = 0; v < plan.nv; ++v, rk.next()) {
            const Visit x = plan.at(v, bifocal);
            const int st = rk.s;
            mbar_wait(&bars->k_full[st], rk.ph);
            if (x.mode == 2) {
                if (v == plan.n_local) {                              // first remote visit: Q -> Q' = R(Delta q) Q
                    if (plan.n_local > 0) mbar_wait(&bars->q_local_done, 0);
                    tc_fence_after();
                    stage_q_rot(qrow, valid, valid ? q : 0, p.G, p.lo, p.hi, tmem + lane_base + TM_QA, tmem + lane_base + TM_QB, precise, p.selinfo + kvh * 16);
                    tmem_st_wait();
                    tc_fence_before();
                }
                if (!p.prerot) {
                    rotate_k_rows<RR, KBOX>(smem_u32(sK(st)), smem_u32(sKl(st)), (unsigned)(x.kt * BN + 64 * cta), rot, precise);
                    fence_proxy_async_smem();
                    if (x.kt > 0) rot.prefetch((unsigned)((x.kt - 1) * BN + 64 * cta));   // next remote visit's first row
                }
            }
            __syncwarp();
            if (lane == 0) {
                if (x.mode == 2 && v == plan.n_local) arrive_leader(&bars->q_rot_done);
                arrive_leader(&bars->k_ready[st]);
            }
        }
    } else if (warp >= 4 && warp < 12) {
        // ===================== softmax groups (steps a6-a8) =====================
        // Two threads per query row: warps w and w+4 hold the same 32 rows, column half `half` (64 keys) each.
        // The S values are loaded ONCE into registers; the row max is combined through shared memory.
        const int half = (warp - 4) >> 2;
        const int quad = warp & 3;
        const int r = (quad << 5) | lane;
        const uint32_t lane_base = (uint32_t)(quad << 5) << 16;
        const uint32_t tO = tmem + lane_base + TM_O + 64 * half;
        const float sl2 = (1.0f / sqrtf((float)D)) * kLog2e;
        const uint64_t sl2x2 = pack2(sl2, sl2);
        float m_ref = -INFINITY;
        uint64_t l2a = 0, l2b = 0;                                     // packed fp32x2 partial row sums
        for (int v = 0; v < plan.nv; ++v) {
            const Visit x = plan.at(v, bifocal);
            const uint32_t tS = tmem + lane_base + TM_S + (v & 1) * 128;
            const long long k0 = (long long)x.kt * BN;
            const long long qrel = q0 + r - k0;
            int lo = 0, hi = BN - 1;
            bool masked = false;
            if (x.kt == qb) { hi = (int)qrel; masked = true; }                                    // causal diagonal
            if (x.mode == 1 && (q0 + BM - 1 - k0 > p.w0)) {                                      // q-k <= w0 (R1)
                const long long a = qrel - p.w0;
                lo = a > 0 ? (int)a : 0;
                masked = true;
            }
            if (x.mode == 2 && (q0 - (k0 + BN - 1) <= p.w0)) {                                   // q-k > w0
                const long long a = qrel - p.w0 - 1;
                hi = a < hi ? (int)a : hi;
                masked = true;
            }
            lo -= 64 * half; hi -= 64 * half;                          // in this thread's 64 columns
            mbar_wait(&bars->s_full[v & 1], (v >> 1) & 1);
            tc_fence_after();
            uint32_t sa[32], sb[32];
            tmem_ld32(tS + 64 * half, sa);
            tmem_ld32(tS + 64 * half + 32, sb);
            tmem_ld_wait();
            if (masked) {
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    if (j < lo || j > hi) sa[j] = 0xff800000u;         // -inf: exp2 -> 0, never wins the max
                    if (j + 32 < lo || j + 32 > hi) sb[j] = 0xff800000u;
                }
            }
            float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
#pragma unroll
            for (int j = 0; j < 32; j += 8) {
                mx0 = max3(mx0, __uint_as_float(sa[j]), __uint_as_float(sa[j + 1]));
                mx1 = max3(mx1, __uint_as_float(sa[j + 2]), __uint_as_float(sa[j + 3]));
                mx2 = max3(mx2, __uint_as_float(sa[j + 4]), __uint_as_float(sa[j + 5]));
                mx3 = max3(mx3, __uint_as_float(sa[j + 6]), __uint_as_float(sa[j + 7]));
                mx0 = max3(mx0, __uint_as_float(sb[j]), __uint_as_float(sb[j + 1]));
                mx1 = max3(mx1, __uint_as_float(sb[j + 2]), __uint_as_float(sb[j + 3]));
                mx2 = max3(mx2, __uint_as_float(sb[j + 4]), __uint_as_float(sb[j + 5]));
                mx3 = max3(mx3, __uint_as_float(sb[j + 6]), __uint_as_float(sb[j + 7]));
            }
            float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
            xchg[((v & 1) * 2 + half) * BM + r] = mx;
            named_bar_sync(1 + quad, 64);                              // the two warps of this row quadrant
            mx = fmaxf(mx, xchg[((v & 1) * 2 + (half ^ 1)) * BM + r]);
            const float mnew = mx * sl2;
            if (v == 0) {
                m_ref = mnew;
            } else {
                const bool need = mnew > m_ref + 8.0f;                 // lazy rescale: only on a jump of 2^8
                if (__any_sync(0xffffffffu, need)) {
                    mbar_wait(&bars->pv_done, (v - 1) & 1);            // O += P V of visit v-1 must have landed
                    tc_fence_after();
                    const float alpha = need ? ex2(m_ref - mnew) : 1.0f;
                    if (need) m_ref = mnew;
                    const uint64_t al2 = pack2(alpha, alpha);
                    l2a = fmul2(l2a, al2); l2b = fmul2(l2b, al2);
                    uint32_t rg[16];
#pragma unroll 1
                    for (int ch = 0; ch < 4; ++ch) {
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
            if (masked) exp_block<false>(sa, sl2x2, mneg2, l2a, l2b, pk); else exp_block<true>(sa, sl2x2, mneg2, l2a, l2b, pk);
            tmem_st16(tS + 32 * half, pk);
            if (masked) exp_block<false>(sb, sl2x2, mneg2, l2a, l2b, pk); else exp_block<true>(sb, sl2x2, mneg2, l2a, l2b, pk);
            tmem_st16(tS + 32 * half + 16, pk);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) arrive_leader(&bars->p_full[v & 1]);
        }
        // ---- epilogue (step a8) ----
        float la, lb, lc, ld;
        unpack2(l2a, la, lb); unpack2(l2b, lc, ld);
        float l = (la + lb) + (lc + ld);
        xchg[(2 + half) * BM + r] = l;                                 // slot parity 1 of the last visit's pair is free:
        named_bar_sync(1 + quad, 64);                                  //   (nv-1)&1 may be 1, so use a dedicated sync
        l += xchg[(2 + (half ^ 1)) * BM + r];
        mbar_wait(&bars->o_full, 0);
        tc_fence_after();
        const long long q = q0 + r;
        const float inv = 1.0f / l;
        const bool qok = q >= 0 && q < p.L;
        __nv_bfloat16* orow = p.out + ((size_t)(qok ? q : 0) * p.H_q + head) * D + 64 * half;
#pragma unroll
        for (int ch = 0; ch < 2; ++ch) {
            uint32_t rg[32];
            tmem_ld32(tO + ch * 32, rg);
            tmem_ld_wait();
            if (qok) {
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
        if (half == 0 && qok) p.lse[(size_t)head * p.L + q] = (m_ref + log2f(l)) * 0.6931471805599453f;
    }
    tc_fence_before();
    cluster_sync_all();                                            // the peer may still be reading our smem / TMEM
    if (warp == W_MMA) tmem_dealloc2<512>(tmem);
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                    const __grid_constant__ CUtensorMap tmKh, const __grid_constant__ CUtensorMap tmKe,
                    const __grid_constant__ CUtensorMap tmKl, const Params p) {
    prefill_body(tmK, tmV, tmKh, tmKe, tmKl, p);
}

// ---- 8(f)-1: rotate K once into a scratch (the workspace variant) -------------------------------------------
// K'hi [L, H_kv, 128] fp16, K'e5 [L, H_kv, 128] e5m2 (K' rounded), K'lo [L, H_kv, 128] e5m2 (K' - K'hi): exactly the
// three operands the rotate group otherwise produces per visit.  Thread = (key k, KV head, 16-byte chunk c).
// Pair energies for the selective compensation.  The sequence is cut into gridDim.x contiguous blocks of rows; a CTA
// measures the MEAN energy x_i^2 + x_{i+64}^2 of every pair i over (a sample of) its block and head h, and the table keeps
// the MAXIMUM over blocks (and over the query heads of a KV group): e[(h / gdiv) * 64 + i] = max_blocks mean_rows(...).
// A global mean (round 1) cannot see a channel that is loud in only part of the sequence; the block maximum can, and
// for stationary inputs it equals the mean up to sampling noise (blocks hold >= 1024 rows).
// grid (blocks, H), 256 threads: pair i = t & 63, row lane t >> 6.  Energies are >= 0, so their bit patterns order as ints.
__global__ void __launch_bounds__(256) pair_energy_kernel(const __nv_bfloat16* __restrict__ X, float* __restrict__ e,
                                                          long long L, int H, int gdiv, int stride) {
    __shared__ float red[256];
    const int i = threadIdx.x & 63, sub = threadIdx.x >> 6, h = blockIdx.y;
    const long long R = (L + gridDim.x - 1) / gridDim.x;
    const long long r0 = (long long)blockIdx.x * R, r1 = r0 + R < L ? r0 + R : L;
    float acc = 0.f;
    for (long long k = r0 + (long long)sub * stride; k < r1; k += 4ll * stride) {
        const __nv_bfloat16* r = X + ((size_t)k * H + h) * D;
        const float x1 = __bfloat162float(r[i]), x2 = __bfloat162float(r[i + 64]);
        acc += x1 * x1 + x2 * x2;
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    if (sub == 0 && r1 > r0) {
        const float n = (float)((r1 - r0 + stride - 1) / stride);
        const float m = (red[i] + red[64 + i] + red[128 + i] + red[192 + i]) / n;
        atomicMax(reinterpret_cast<int*>(&e[(h / gdiv) * 64 + i]), __float_as_int(m));
    }
}

// Per KV head: weight w_i = (block-max pair energy of K) x (of Q); in every chunk of 8 pairs the two heaviest are
// compensated (PRMT selector j0 | j1 << 4).  The pairs left out add rounding noise of about
// sigma = scale * 2^-10 / (1.44 sqrt(12)) * sqrt(sum of their w_i) to a remote score.  The head falls back to
// the full e5m2 cross terms (flag at [8]) when sigma > SEL_SIGMA_MAX, or when a pair that was left out is LOUD -- more
// than SEL_LOUD times the mean weight of the pairs left out (three outlier pairs in one chunk; measured: one such pair
// alone puts the lse error at 2e-3).
constexpr float SEL_SIGMA_MAX = 3.0e-4f;
constexpr float SEL_LOUD = 4.0f;
constexpr float SEL_COINCIDENT = 100.0f;
__global__ void __launch_bounds__(64) select_pairs_kernel(const float* __restrict__ eK, const float* __restrict__ eQ,
                                                          uint32_t* __restrict__ selinfo) {
    __shared__ float w[64];
    __shared__ float resid[8], loud[8], selmax[8];
    __shared__ float med;
    const int kvh = blockIdx.x, t = threadIdx.x;
    w[t] = eK[kvh * 64 + t] * eQ[kvh * 64 + t];
    __syncthreads();
    {                                                                 // median weight of the 64 pairs (rank 32, ties by index)
        int rank = 0;
        for (int j = 0; j < 64; ++j) rank += (w[j] < w[t] || (w[j] == w[t] && j < t)) ? 1 : 0;
        if (rank == 32) med = w[t];
    }
    if (t < 8) {
        int j0 = 0;
        for (int j = 1; j < 8; ++j) if (w[8 * t + j] > w[8 * t + j0]) j0 = j;
        int j1 = j0 == 0 ? 1 : 0;
        for (int j = 0; j < 8; ++j) if (j != j0 && w[8 * t + j] > w[8 * t + j1]) j1 = j;
        float r = 0.f, mx = 0.f;
        for (int j = 0; j < 8; ++j) if (j != j0 && j != j1) { r += w[8 * t + j]; mx = fmaxf(mx, w[8 * t + j]); }
        resid[t] = r;
        loud[t] = mx;
        selmax[t] = fmaxf(w[8 * t + j0], w[8 * t + j1]);
        const int a = j0 < j1 ? j0 : j1, b = j0 < j1 ? j1 : j0;
        selinfo[kvh * 16 + t] = (uint32_t)(a | (b << 4));
    }
    __syncthreads();
    if (t == 0) {
        float r = 0.f, mx = 0.f;
        for (int c = 0; c < 8; ++c) { r += resid[c]; mx = fmaxf(mx, loud[c]); }
        const float sigma = rsqrtf((float)D) * 1.96e-4f * sqrtf(r);
        const bool full = sigma > SEL_SIGMA_MAX || !(sigma == sigma) || mx > SEL_LOUD * (r / 48.0f);
        selinfo[kvh * 16 + 8] = full ? 1u : 0u;
        // A SELECTED pair that is loud in Q and in K at once: its cross terms are large and e5m2 (3 significant bits) leaves 17 %
        // of them (measured: lse 1.6e-3 at Q x2 . K x8, weight 256 x the median; 2.8e-4 at K x8 alone, 64 x).  The two-tile
        // kernel then keeps the selected pairs' cross terms in fp16 (prefill_umma2.cu, precise 4).
        float sm = 0.f;
        for (int c = 0; c < 8; ++c) sm = fmaxf(sm, selmax[c]);
        selinfo[kvh * 16 + 9] = (sm > SEL_COINCIDENT * med) ? 1u : 0u;
    }
}

__global__ void __launch_bounds__(256) prerotate_k_kernel(const __nv_bfloat16* __restrict__ K, __half* __restrict__ Kh,
                                                          unsigned char* __restrict__ Ke, unsigned char* __restrict__ Kl,
                                                          long long L, int H_kv, long long G,
                                                          const float2* __restrict__ lo, const float2* __restrict__ hi,
                                                          const uint32_t* __restrict__ selinfo) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= L * H_kv * 8) return;
    const int c = (int)(idx & 7);
    const long long row = idx >> 3;                                   // k * H_kv + kvh
    const long long k = row / H_kv;
    const uint4 u1 = __ldg(reinterpret_cast<const uint4*>(K + row * D) + c);
    const uint4 u2 = __ldg(reinterpret_cast<const uint4*>(K + row * D) + 8 + c);
    float cs_c[8], cs_s[8];
    cs8(lo, hi, k, G, 8 * c, cs_c, cs_s);
    const uint32_t a[4] = {u1.x, u1.y, u1.z, u1.w}, b[4] = {u2.x, u2.y, u2.z, u2.w};
    uint32_t h1[4], h2[4], l1[4], l2[4];
    rot8(a, b, cs_c, cs_s, h1, h2, l1, l2);
    reinterpret_cast<uint4*>(Kh + row * D)[c] = make_uint4(h1[0], h1[1], h1[2], h1[3]);
    reinterpret_cast<uint4*>(Kh + row * D)[8 + c] = make_uint4(h2[0], h2[1], h2[2], h2[3]);
    const uint2 eh1 = make_uint2(e5m2x4(h1[0], h1[1]), e5m2x4(h1[2], h1[3])), eh2 = make_uint2(e5m2x4(h2[0], h2[1]), e5m2x4(h2[2], h2[3]));
    const uint2 el1 = make_uint2(e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3])), el2 = make_uint2(e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]));
    const int kvh = (int)(row - k * H_kv);
    if (selinfo != nullptr && selinfo[kvh * 16 + 8] == 0u) {
        // selective mode: one 128-byte row per key = region LO (32 B) | region HI (32 B) | unused; chunk c of a region is
        // [x1(f0) x1(f1) x2(f0) x2(f1)], the layout rotate_rows2 (rot.cuh) writes on the fly
        const uint32_t sj = selinfo[kvh * 16 + c];
        uint32_t* dst = reinterpret_cast<uint32_t*>(Ke + row * D);
        dst[c] = (__byte_perm(el1.x, el1.y, sj) & 0xffffu) | (__byte_perm(el2.x, el2.y, sj) << 16);
        dst[8 + c] = (__byte_perm(eh1.x, eh1.y, sj) & 0xffffu) | (__byte_perm(eh2.x, eh2.y, sj) << 16);
    } else {
        reinterpret_cast<uint2*>(Ke + row * D)[c] = eh1;
        reinterpret_cast<uint2*>(Ke + row * D)[8 + c] = eh2;
        reinterpret_cast<uint2*>(Kl + row * D)[c] = el1;
        reinterpret_cast<uint2*>(Kl + row * D)[8 + c] = el2;
    }
}

// Eq.(7) P:114 with the minus sign: O = (W_A O_A + W_B O_B - W_C O_C) / (W_A + W_B - W_C), W_X = exp(l_X - M); numerator and
// denominator in fp32.  The partial outputs are fp32; the result is rounded once to bf16.  Thread = (row q, head h,
// 8 channels); lA is read from and the merged lse written to `lse`.
__global__ void __launch_bounds__(256) merge_abc_kernel(__nv_bfloat16* __restrict__ out, float* __restrict__ lse,
                                                        const float* __restrict__ oA, const float* __restrict__ oB,
                                                        const float* __restrict__ lB, const float* __restrict__ oC,
                                                        const float* __restrict__ lC, long long L, int H_q) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= L * H_q * 16) return;
    const int c = (int)(idx & 15);
    const long long row = idx >> 4;                                   // q * H_q + h
    const long long q = row / H_q;
    const int h = (int)(row - q * H_q);
    const size_t li = (size_t)h * L + q;
    const float a = lse[li], b = lB[li], cc = lC[li];
    const float M = fmaxf(a, b);
    const float wA = __expf(a - M), wB = __expf(b - M), wC = __expf(cc - M);
    const float den = wA + wB - wC;
    const float inv = 1.0f / den;
    float va[8], vb[8], vc[8];
    *reinterpret_cast<float4*>(va) = reinterpret_cast<const float4*>(oA + row * D)[2 * c];
    *reinterpret_cast<float4*>(va + 4) = reinterpret_cast<const float4*>(oA + row * D)[2 * c + 1];
    *reinterpret_cast<float4*>(vb) = reinterpret_cast<const float4*>(oB + row * D)[2 * c];
    *reinterpret_cast<float4*>(vb + 4) = reinterpret_cast<const float4*>(oB + row * D)[2 * c + 1];
    *reinterpret_cast<float4*>(vc) = reinterpret_cast<const float4*>(oC + row * D)[2 * c];
    *reinterpret_cast<float4*>(vc + 4) = reinterpret_cast<const float4*>(oC + row * D)[2 * c + 1];
    uint32_t w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
        w[j] = bf16x2((wA * va[2 * j] + wB * vb[2 * j] - wC * vc[2 * j]) * inv,
                      (wA * va[2 * j + 1] + wB * vb[2 * j + 1] - wC * vc[2 * j + 1]) * inv);
    reinterpret_cast<uint4*>(out + row * D)[c] = make_uint4(w[0], w[1], w[2], w[3]);
    __syncwarp();                                                     // the 16 threads of a (q, h) all read lse first
    if (c == 0) lse[li] = M + __logf(den);
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(sym);
    }
    return fn;
}

// [L, H, 128] bf16 tensor seen as (d, H, L); box = 64 channels x 1 head x `rows` rows, SWIZZLE_128B, OOB rows -> 0
// bytes = 1: the same tensor with one-byte elements (the e5m2 copies), box = 128 channels x 1 head x `rows` rows
static bool make_tensor_map(CUtensorMap* m, const void* base, long long L, int H, int rows, int bytes) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)H, (cuuint64_t)L};
    cuuint64_t strides[2] = {(cuuint64_t)D * bytes, (cuuint64_t)H * D * bytes};
    cuuint32_t box[3] = {(cuuint32_t)(128 / bytes), 1, (cuuint32_t)rows};
    cuuint32_t es[3] = {1, 1, 1};
    return fn(m, bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// pair energies of K (every row) and Q (every 8th row) and the per-head selection table (selective compensation);
// scratch: eK [H_kv][64] | eQ [H_kv][64] floats, then selinfo [H_kv][16] uint32
static size_t selection_bytes(int H_kv) { return align256((size_t)H_kv * 64 * 4 * 2) + align256((size_t)H_kv * 16 * 4); }
static int run_selection(const void* Q, const void* K, long long L, int H_q, int H_kv, unsigned char* scratch,
                         cudaStream_t st, uint32_t** selinfo_out) {
    float* eK = reinterpret_cast<float*>(scratch);
    float* eQ = eK + (size_t)H_kv * 64;
    uint32_t* selinfo = reinterpret_cast<uint32_t*>(scratch + align256((size_t)H_kv * 64 * 4 * 2));
    if (cudaMemsetAsync(eK, 0, (size_t)H_kv * 64 * 4 * 2, st) != cudaSuccess) return check_launch("memset");
    // blocks of >= 1024 rows (at most 64 of them): the block mean then carries ~3 % of sampling noise, so the maximum over
    // blocks of a stationary input stays within ~10 % of its mean; K is read in full, Q every 8th row
    const int sk = 1, sq = 8;
    long long nb = L / 1024;
    nb = nb < 1 ? 1 : nb > 64 ? 64 : nb;
    pair_energy_kernel<<<dim3((unsigned)nb, H_kv), 256, 0, st>>>((const __nv_bfloat16*)K, eK, L, H_kv, 1, sk);
    pair_energy_kernel<<<dim3((unsigned)nb, H_q), 256, 0, st>>>((const __nv_bfloat16*)Q, eQ, L, H_q, H_q / H_kv, sq);
    select_pairs_kernel<<<H_kv, 64, 0, st>>>(eK, eQ, selinfo);
    note_launch(3);
    *selinfo_out = selinfo;
    return check_launch("select_pairs_kernel");
}

bool make_kv_tensor_map(CUtensorMap* m, const void* base, long long L, int H, int rows) {
    return make_tensor_map(m, base, L, H, rows, 2);
}

size_t umma_prefill_prerot_workspace_bytes(long long L, int H_kv, int d);
size_t umma_prefill_unfused_workspace_bytes(long long L, int H_q, int H_kv, int d) {
    const size_t nq = (size_t)L * H_q * d;
    // the workspace variant's region (tables | K'hi fp16 | K' / K'lo e5m2 | selection) | O_A, O_B, O_C fp32 | lse_B | lse_C
    return umma_prefill_prerot_workspace_bytes(L, H_kv, d) + 3 * align256(4 * nq) + 2 * align256((size_t)L * H_q * 4);
}

// 1: the default precision of the on-the-fly two-tile kernel uses the selective e5m2 compensation; 0: the full cross terms
constexpr int g_otf_selective = 1;

bool umma_prefill_supported(long long L, int H_q, int H_kv, int d, int dtype) {
    if (dtype != JETLONG_BF16 || d != 128 || H_kv < 1 || H_q % H_kv) return false;
    return L >= 1 && L < (1ll << 30);                // any GQA group size: odd groups (MHA included) run a lone-head unit per group
}

size_t umma_prefill_workspace_bytes(long long L, int, int H_kv, int d) { return two_level_bytes(L + 256, d) + selection_bytes(H_kv); }

// pre-rotated variant: tables, then K'hi (fp16), K' (e5m2), K'lo (e5m2), each [L, H_kv, 128]
size_t umma_prefill_prerot_workspace_bytes(long long L, int H_kv, int d) {
    const size_t n = (size_t)L * H_kv * d;
    return two_level_bytes(L + 256, d) + align256(2 * n) + 2 * align256(n) + selection_bytes(H_kv);
}

int launch_prefill_umma(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                        int H_kv, int d, long long w0, long long G, double theta, bool bifocal, int precise, void* ws,
                        size_t ws_bytes, cudaStream_t st, bool prerot, bool g_two_tile, FreqMap fm, int qb_lo, int qb_hi,
                        long long L_sel) {
    (void)ws_bytes;
    CUtensorMap tmK, tmV;
    if (!make_kv_tensor_map(&tmK, K, L, H_kv, 64) || !make_kv_tensor_map(&tmV, V, L, H_kv, 128)) return JETLONG_UNSUPPORTED;
    Params p;
    p.Q = (const __nv_bfloat16*)Q;
    p.out = (__nv_bfloat16*)out;
    p.lse = lse;
    p.L = L; p.w0 = w0; p.G = G;
    p.H_q = H_q; p.H_kv = H_kv; p.g = H_q / H_kv;
    p.bifocal = bifocal ? 1 : 0;
    const bool full_e5m2 = precise == 6;                           // JETLONG_PRECISION_COMPENSATED_E5M2: never the selective form
    if (full_e5m2) precise = 2;
    p.precise = precise;
    p.prerot = 0;
    p.window_only = 0;
    p.qk_f16 = 0;
    p.selinfo = nullptr;
    p.qb_top = (int)((L + BM - 1) / BM);
    p.qb_lo = 0;
    CUtensorMap tmKh = tmK, tmKe = tmK, tmKl = tmK;
    p.lo = nullptr; p.hi = nullptr;
    if (bifocal) {
        int rc = build_two_level(ws, L + 256, d, theta, st, fm);
        if (rc != JETLONG_OK) return rc;
        p.lo = reinterpret_cast<const float2*>((unsigned char*)ws + 256);
        p.hi = p.lo + 256 * (d / 2);
        if (prerot) {
            // the scratch holds e5m2 cross-term operands only: the fp16 mode is served by the full e5m2 terms (2),
            // the default by the selective e5m2 terms (3) with a per-head fallback to 2
            // (the one-tile kernels of this file read the full e5m2 operands only)
            precise = p.precise = (precise == 0 ? 0 : (precise == 1 || full_e5m2 || !g_two_tile) ? 2 : 3);
            const size_t n = (size_t)L * H_kv * d;
            unsigned char* base = (unsigned char*)ws + two_level_bytes(L + 256, d);
            __half* Kh = reinterpret_cast<__half*>(base);
            unsigned char* Ke = base + align256(2 * n);
            unsigned char* Kl = Ke + align256(n);
            uint32_t* selinfo = nullptr;
            if (precise == 3) {
                rc = run_selection(Q, K, L, H_q, H_kv, Kl + align256(n), st, &selinfo);
                if (rc != JETLONG_OK) return rc;
                p.selinfo = selinfo;
            }
            const long long items = L * H_kv * 8;
            prerotate_k_kernel<<<(unsigned)((items + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)K, Kh, Ke, Kl, L, H_kv, G,
                                                                               p.lo, p.hi, selinfo);
            note_launch();
            rc = check_launch("prerotate_k_kernel");
            if (rc != JETLONG_OK) return rc;
            if (!make_tensor_map(&tmKh, Kh, L, H_kv, 64, 2) || !make_tensor_map(&tmKe, Ke, L, H_kv, 64, 1) ||
                !make_tensor_map(&tmKl, Kl, L, H_kv, 64, 1))
                return JETLONG_UNSUPPORTED;
            p.prerot = 1;
        } else if (precise == 2 && g_otf_selective && !full_e5m2 && g_two_tile) {
            // on the fly, default precision: selective e5m2 compensation as in the workspace variant (per-head fallback
            // to the full cross terms inside the kernel)
            uint32_t* selinfo = nullptr;
            // L_sel: the rows the selection statistics may read (jetlong_prefill_host launches row chunks while later rows
            // are still being uploaded)
            rc = run_selection(Q, K, L_sel > 0 && L_sel < L ? L_sel : L, H_q, H_kv, (unsigned char*)ws + two_level_bytes(L + 256, d), st, &selinfo);
            if (rc != JETLONG_OK) return rc;
            p.selinfo = selinfo;
            precise = p.precise = 3;
        }
    }
    if ((H_q / H_kv) & 1) {                          // odd group sizes exist only in the two-tile kernel
        g_two_tile = true;
        if (precise == 1) precise = p.precise = 2;
    }
    if (g_two_tile && prefill_v2_serves(precise)) {
        PrefillV2Args a;
        if (!make_kv_tensor_map(&a.tmQ, Q, L, H_q, 128)) return JETLONG_UNSUPPORTED;
        a.tmK = tmK; a.tmV = tmV; a.tmKh = tmKh; a.tmKe = tmKe; a.tmKl = tmKl;
        a.out = p.out; a.lse = lse; a.L = L; a.w0 = w0; a.G = G; a.H_q = H_q; a.H_kv = H_kv;
        a.bifocal = p.bifocal; a.precise = precise; a.prerot = p.prerot; a.window_only = 0; a.qk_f16 = 0; a.out_f32 = 0;
        a.lo = p.lo; a.hi = p.hi; a.selinfo = p.selinfo;
        a.qb_lo = qb_lo; a.qb_hi = qb_hi;
        return launch_prefill_v2(a, st);
    }
    if (qb_lo != 0 || qb_hi >= 0) return JETLONG_UNSUPPORTED;        // row chunks exist only in the two-tile kernel
    if (cudaFuncSetAttribute(prefill_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess)
        return check_launch("prefill_umma attr");
    const int n_qb = (int)((L + BM - 1) / BM);
    const unsigned grid = 2u * (unsigned)n_qb * (unsigned)(H_q / 2);
    prefill_umma_kernel<<<grid, NTHREADS, SMEM_BYTES, st>>>(tmK, tmV, tmKh, tmKe, tmKl, p);
    note_launch();
    return check_launch("prefill_umma_kernel");
}

}  // namespace jetlong


namespace jetlong {

// ---- 8(f)-2: the unfused three-call baseline ("Jet-Long (unfused)") ---------------------------------------
// Three launches of the two-tile kernel, each returning (O_X fp32, l_X), then Eq.(7) with the minus sign:
//   A = the local band 0 <= q-k <= w0 on the stored Q, K;
//   B = full causal attention at the remote positions: the bifocal kernel with an EMPTY local window (w0 = -1), remote
//       operands from the workspace variant's scratch, compensated exactly as the fused product;
//   C = the band scored with the remote operands (window_only = 2).
// Round 1 ran B and C on once-rounded fp16 operands and stored O_B, O_C in bf16 (lse ~3e-3, out errors up to 0.9 from the
// cancellation); with fp32 partials and the product's compensated operands the baseline is as accurate as the fused
// kernel up to the cancellation Eq.(7) itself carries.
int launch_prefill_unfused(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                           int H_kv, int d, long long w0, long long G, double theta, void* ws, cudaStream_t st) {
    int rc = build_two_level(ws, L + 256, d, theta, st);
    if (rc != JETLONG_OK) return rc;
    const float2* lo = reinterpret_cast<const float2*>((unsigned char*)ws + 256);
    const float2* hi = lo + 256 * (d / 2);
    const size_t nq = (size_t)L * H_q * d, nk = (size_t)L * H_kv * d;
    unsigned char* base = (unsigned char*)ws + two_level_bytes(L + 256, d);
    __half* Kh = reinterpret_cast<__half*>(base);
    unsigned char* Ke = base + align256(2 * nk);
    unsigned char* Kl = Ke + align256(nk);
    uint32_t* selinfo = nullptr;
    rc = run_selection(Q, K, L, H_q, H_kv, Kl + align256(nk), st, &selinfo);
    if (rc != JETLONG_OK) return rc;
    prerotate_k_kernel<<<(unsigned)((L * H_kv * 8 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)K, Kh, Ke, Kl, L, H_kv, G, lo, hi, selinfo);
    note_launch();
    if ((rc = check_launch("prerotate_k_kernel")) != JETLONG_OK) return rc;
    unsigned char* part = (unsigned char*)ws + umma_prefill_prerot_workspace_bytes(L, H_kv, d);
    float* oA = reinterpret_cast<float*>(part);
    float* oB = reinterpret_cast<float*>(part + align256(4 * nq));
    float* oC = reinterpret_cast<float*>(part + 2 * align256(4 * nq));
    float* lB = reinterpret_cast<float*>(part + 3 * align256(4 * nq));
    float* lC = reinterpret_cast<float*>(reinterpret_cast<unsigned char*>(lB) + align256((size_t)L * H_q * 4));
    PrefillV2Args a;
    if (!make_kv_tensor_map(&a.tmK, K, L, H_kv, 64) || !make_kv_tensor_map(&a.tmV, V, L, H_kv, 128) ||
        !make_kv_tensor_map(&a.tmQ, Q, L, H_q, 128) || !make_tensor_map(&a.tmKh, Kh, L, H_kv, 64, 2) ||
        !make_tensor_map(&a.tmKe, Ke, L, H_kv, 64, 1) || !make_tensor_map(&a.tmKl, Kl, L, H_kv, 64, 1))
        return JETLONG_UNSUPPORTED;
    a.L = L; a.G = G; a.H_q = H_q; a.H_kv = H_kv; a.bifocal = 1; a.precise = 3; a.qk_f16 = 0; a.out_f32 = 1;
    a.lo = lo; a.hi = hi; a.selinfo = selinfo;
    a.out = oA; a.lse = lse; a.w0 = w0; a.prerot = 0; a.window_only = 1;                         // A
    if ((rc = launch_prefill_v2(a, st)) != JETLONG_OK) return rc;
    a.out = oB; a.lse = lB; a.w0 = -1; a.prerot = 1; a.window_only = 0;                          // B
    if ((rc = launch_prefill_v2(a, st)) != JETLONG_OK) return rc;
    a.out = oC; a.lse = lC; a.w0 = w0; a.prerot = 1; a.window_only = 2;                          // C
    if ((rc = launch_prefill_v2(a, st)) != JETLONG_OK) return rc;
    merge_abc_kernel<<<(unsigned)((L * H_q * 16 + 255) / 256), 256, 0, st>>>((__nv_bfloat16*)out, lse, oA, oB, lB, oC, lC, L, H_q);
    note_launch();
    return check_launch("merge_abc_kernel");
}

}  // namespace jetlong
