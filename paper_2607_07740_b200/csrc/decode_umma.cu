// decode_umma.cu -- tcgen05 split-KV batch-1 decode for bf16, head_dim 128, up to 16 query heads per KV head
// (steps a9, a7, a8).  HBM-bound scan: the KV cache is streamed once, by TMA, at full bandwidth; nothing but the
// correction rotation of remote keys touches the ALUs per cache element.
//
// A CTA owns one KV head and a contiguous key range.  Per 128-key tile (KEYS on the UMMA M axis):
//   S^T[key, head] = K[key, :] . Q[head, :]        UMMA M=128 (keys), N=16 (heads, zero padded), K=128 (channels)
//   P[head, key]   = exp2(S^T * scale*log2e - m)   one thread per key, 16 values each
//   O^T[ch, head] += V^T[ch, key] . P[head, key]   UMMA M=128 (channels), N=16, K=128 (keys); A = V tile, MN-major
// Remote tiles (k < L-1-w0): the rotate group turns the TMA-loaded K tile into K' = R(Delta k) K in shared memory
// (fp32 rotate, fp16 hi in place + fp16 lo in a side buffer), Q' = R(Delta q) Q is prepared once per CTA, and
// S^T = K'hi Q'hi + K'lo Q'hi + K'hi Q'lo (compensated; the MMAs are ~free here).  The cache is only read.
// S^T = K'hi [Q'hi; Q'lo] (fp16, one pass over the K tile, N = 32) + K'lo Q'hi (e5m2, kind::f8f6f4).
// Warp roles (480 threads): warp 0 K producer (TMA), warp 1 MMA issuer, warp 2 V producer (TMA), warps 3-10 rotate
// group, warps 11-14 softmax.
// Partial (m, l, O) states go to the workspace and are merged by decode_merge_kernel (additive LSE merge).
#include <cuda.h>
#include <math.h>

#include "common.cuh"
#include "umma.cuh"
#include "rot.cuh"

namespace jetlong {

namespace {

using namespace ptx;
using namespace dev;

constexpr int D = 128, BN = 128;
constexpr int NH = 16;                               // UMMA N: query heads of one KV group, zero padded
constexpr int KS = 3, VS = 2;                        // K / V ring depths; a K stage is K (hi in place) | K lo (e5m2)
constexpr int BOXB = BN * 128;                       // one SWIZZLE_128B box: 128 rows x 128 B = 16 KB
constexpr int TILE = 2 * BOXB;                       // 32 KB (channels 0-63 | 64-127)
constexpr int KSTAGE = TILE + BOXB;                  // K tile + its e5m2 lo copy [128 rows][128 B]: 48 KB
constexpr int QBUF = 2 * NH * 128;                   // [2 boxes][16 rows][128 B] = 4 KB (raw Q, P)
constexpr int QCBUF = 2 * 2 * NH * 128;              // [2 boxes][32 rows][128 B] = 8 KB: rows 0-15 Q'hi, rows 16-31 Q'lo
constexpr int QYBUF = NH * 128;                      // [16 rows][128 B] = 2 KB: Q'hi as e5m2
constexpr int RW = 8;                                // rotate warps
constexpr int RT = RW * 32;                          // rotate threads
constexpr int RROWS = 1024 / RT;                     // key rows per rotate thread (8 chunks x 128 rows / RT)
constexpr int NTHREADS = 96 + RT + 128;             // warps: 0 K producer, 1 MMA, 2 V producer, 3.. rotate, last 4 softmax
constexpr float kLog2e = 1.4426950408889634f;
constexpr uint32_t SCOLS = 4 * NH;                   // columns of one S buffer: [hi | lo | d/dn | d2/dn2] blocks of 16 heads
constexpr uint32_t TM_S = 0, TM_O = 2 * SCOLS;       // S0 | S1 (64 fp32 columns each, see issue_s) | O (16)
constexpr int TM_COLS = 256;

struct Bars {
    uint64_t k_full[KS], k_ready[KS], k_empty[KS];
    uint64_t v_full[VS], v_empty[VS];
    uint64_t s_full[2], p_full[2];
    uint64_t pv_done, o_full, q_ready;
    uint32_t tmem_base;
    float red[4 * NH];                               // cross-warp max / sum exchange of the softmax group
    uint32_t chk[4];                                 // per-warp partial hashes of the table check (rotate warps 0-3)
};

// smem: K ring (K | K lo e5m2 per stage) | V ring | Q raw | Q' (hi rows | lo rows) | Q'hi e5m2 | P | Bars
constexpr size_t OFF_V = (size_t)KS * KSTAGE, OFF_Q = OFF_V + (size_t)VS * TILE, OFF_P = OFF_Q + QBUF + QCBUF + QYBUF,
                 OFF_BARS = OFF_P + QBUF;
constexpr size_t SMEM_BYTES = OFF_BARS + 1024;       // = 227 KB exactly; the dynamic smem base must be 1024-aligned
static_assert(SMEM_BYTES <= 232448, "shared memory budget");

struct Params {
    const __nv_bfloat16* q;
    float* part;                                     // [nsplit][H_q][D+2]
    long long L, w0, G, kps;                         // kps = keys per split, a multiple of BN
    int H_q, H_kv, g, bifocal;                      // g = query heads per KV head served by THIS launch (<= 16)
    int gq, h0;                                      // heads per KV head in q / the partials, first head of this launch in its group
    const float2* lo;
    const float2* hi;
    double theta;                                    // for the table-header check (see the prologue)
    long long n_hi;                                  // rows of the HI table the host asked the table kernel for
    FreqMap fm;                                      // the remote map the tables must have been built for
    int split;                                       // 1: the slow frequency pairs 32-63 are not rotated per key (see SPLIT below)
};
// batched / paged form: blockIdx.z = sequence b with its own length and group size; the cache is a pool of
// 128-row pages (= the TMA tile) addressed through a page table.  A separate kernel argument: the per-sequence arrays are
// indexed at run time, and folding them into Params (which the kernel copies and edits per sequence) put every field of
// it into local memory (measured: 115 -> 121 us per 128K step).
struct BatchInfo {
    int batch;                                       // 0: the single-sequence call
    const int* page_table;                           // [batch][max_pages] physical page of logical tile kt (device memory)
    int max_pages;
    long long part_stride;                           // floats between the partials of consecutive sequences
    long long Ls[16];
    int Gs[16];
};
constexpr int MAXB = 16;

// byte offset of element (row n, k) in a [2 boxes][16 rows][128 B] SWIZZLE_128B K-major operand (16-bit elements)
template <int ROWS = NH> __device__ __forceinline__ int bop_off(int n, int k) {
    return (k >> 6) * (ROWS * 128) + n * 128 + ((((k & 63) >> 3) ^ (n & 7)) << 4) + (k & 7) * 2;
}

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// OR of `pred` over the `nthreads` threads that meet at named barrier `id`
__device__ __forceinline__ bool bar_red_or(int id, int nthreads, bool pred) {
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %3, 0;\n\t"
        "barrier.red.or.pred q, %1, %2, p;\n\t"
        "selp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(r) : "r"(id), "r"(nthreads), "r"((uint32_t)pred) : "memory");
    return r != 0;
}
__device__ __forceinline__ void sts16(uint32_t a, uint16_t v) { asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"(v) : "memory"); }
__device__ __forceinline__ uint16_t bf16_bits(float f) {
    const __nv_bfloat16 b = __float2bfloat16_rn(f);
    return *reinterpret_cast<const uint16_t*>(&b);
}

// programmatic dependent launch: the kernel starts while its stream predecessor (the table check, or the previous
// step's merge) is still draining; griddep_wait() returns once that grid has completed and its writes are visible
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

constexpr uint32_t IDESC_S_BF16 = idesc_f16(1, 1, 0, 0, BN, NH);
constexpr uint32_t IDESC_S_F16 = idesc_f16(0, 0, 0, 0, BN, NH);
constexpr uint32_t IDESC_S_F16_N32 = idesc_f16(0, 0, 0, 0, BN, 2 * NH);
constexpr uint32_t IDESC_S_E5M2 = idesc_f16(1, 1, 0, 0, BN, NH);  // kind::f8f6f4: format code 1 = e5m2
// Bifocal scan: when the producer issues the load of tile v it also asks the TMA unit to fetch tile v + 1 into L2
// (cp.async.bulk.prefetch.tensor).  A K stage is busy from the issue of its load until the MMAs on the ROTATED tile have
// completed; with three stages and ~3.5 us of load latency under full HBM load that life (latency + rotation) set the
// period per tile.  The prefetched tile's load is an L2 hit, the stage turns over sooner.  Measured at 64K: 55.1 -> 51.6 us
// (distance 1), 53.1 (2), 54.2 (3), 59.7 (4), 65.7 (5); K only 51.6, V only 53.9.  The control does not need it and loses
// with it (45.1 -> 51.0 us at distance 3: more requests in flight than DRAM serves in order), so it is off there.
constexpr int PFK = 1, PFV = 1;
static_assert(PFK <= 1 && PFV <= 1, "the paged producers know the page of tile v + 1 only");
constexpr int RO = 1;                                // SPLIT: rows per thread on the odd rotate warps (the even ones take 4 - RO)
constexpr int SB = 8;                                // rows (heads) per block of the slow pairs' operand: SPLIT serves g <= 8
constexpr uint32_t IDESC_S_BF16_N48 = idesc_f16(1, 1, 0, 0, BN, 6 * SB);
constexpr uint32_t IDESC_PV = idesc_f16(1, 1, 1, 0, D, NH);      // A = V^T (smem, MN-major), B = P (smem, K-major)

// SPLIT (slow pairs through the tensor core on the STORED keys).  The correction rotation of pair i at key row m of a tile
// is Rot(alpha_ref + eps), alpha_ref the angle at the tile's reference row (n_ref = n(k0 + 64)) and
// eps = (n_m - n_ref) a_i, a_i the table's unit-step angle (|a_i| = theta_i).  For i >= 32 and rope_theta >= 4.54e5,
// |eps| <= 64 theta_32 <= 0.095, and  Rot(eps) = (1 - eps^2/2) I + eps J  holds to eps^3/6 <= 1.4e-4 (relative, per pair):
//     q'^T Rot(alpha_ref + eps) k = qt^T k + dn (a J^T qt)^T k + dn^2 (-a^2/2 qt)^T k,   qt = Rot(alpha_ref)^T q',  dn = n_m - n_ref.
// So those pairs need no per-key rotation at all: per tile the rotate group writes 8-row blocks of a bf16 B operand
//     block 0: qt hi | 1: unused | 2: qt lo | 3: (a J^T qt) hi | 4: (a J^T qt) lo | 5: -a^2/2 qt      (8 heads x 32 pairs each;
// hi / lo because one bf16 rounding of a full-size term is 2^-9, and of the first-order term still 64 theta_i 2^-9: with loud
// channels on pair 32 that alone broke the lse tolerance, tests/test_gpu_robustness.py), the MMA warp multiplies the stored
// bf16 K slices by them (N = 48), and the softmax thread of key m adds  S[h] + S[16 + h] + dn (S[24 + h] + S[32 + h] + dn S[40 + h])
// (columns h and 16 + h also receive the fast pairs' K'hi Q'hi and K'hi Q'lo).  The stored keys enter exactly (no fp16
// re-rounding, no e5m2 residual).  The operand lives in the unused bytes of the K stage's own e5m2 box (byte ranges 32-63 and
// 96-127 of each row belong to the unrotated channels): rows 0-47 serve channels 32-47 / 48-63, rows 64-111 channels 96-111 /
// 112-127.  More than 8 query heads per KV head do not fit that space: they keep the per-key rotation of all pairs.

struct DPlan {
    long long ks, ke, re, ls;
    int kt_r0, nr, kt_l0, nl, nv;
    __device__ DPlan(const Params& p, int split) {
        ks = (long long)split * p.kps;
        ke = ks + p.kps < p.L ? ks + p.kps : p.L;
        const long long qpos = p.L - 1;
        const long long kb = (p.bifocal && qpos - p.w0 > 0) ? qpos - p.w0 : 0;     // keys >= kb are local (R1)
        re = ke < kb ? ke : kb;
        ls = ks > kb ? ks : kb;
        kt_r0 = (int)(ks / BN);
        nr = re > ks ? (int)((re - 1) / BN) - kt_r0 + 1 : 0;
        kt_l0 = (int)(ls / BN);
        nl = ke > ls ? (int)((ke - 1) / BN) - kt_l0 + 1 : 0;
        nv = nr + nl;
    }
    __device__ int kt(int v) const { return v < nr ? kt_r0 + v : kt_l0 + (v - nr); }
    __device__ bool remote(int v) const { return v < nr; }
};

template <int NG, bool BATCHED>                      // NG = query heads per KV head, rounded up to a power of two
__global__ void __launch_bounds__(NTHREADS, 1)
decode_umma_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV, const Params p0,
                   const __grid_constant__ BatchInfo bi) {
    // the single-sequence instantiation reads its parameters straight from the constant bank; only the batched one
    // works on an edited copy
    Params pb = p0;
    const int* pages = nullptr;                                        // this sequence's row of the page table
    if (BATCHED) {
        const int b = blockIdx.z;
        pb.L = bi.Ls[b];
        pb.G = bi.Gs[b];
        pb.bifocal = (pb.G > 1 && pb.w0 < pb.L - 1) ? 1 : 0;           // step a2, per sequence
        pb.q = p0.q + (size_t)b * p0.H_q * D;
        pb.part = p0.part + (size_t)b * bi.part_stride;
        const long long tiles = (pb.L + BN - 1) / BN, tps = (tiles + gridDim.x - 1) / gridDim.x;
        pb.kps = tps * BN;
        pages = bi.page_table + (size_t)b * bi.max_pages;
    }
    const Params& p = BATCHED ? pb : p0;
    extern __shared__ __align__(1024) unsigned char smem[];
    if ((smem_u32(smem) & 1023u) != 0) __trap();               // SWIZZLE_128B operands need the 1024-byte alignment
    unsigned char* sQ = smem + OFF_Q;                              // raw | hi | lo
    unsigned char* sP = smem + OFF_P;
    Bars* bars = reinterpret_cast<Bars*>(smem + OFF_BARS);
    auto sK = [&](int s) { return smem + (size_t)s * KSTAGE; };                  // K lo (e5m2) of the stage sits at + TILE
    auto sV = [&](int s) { return smem + OFF_V + (size_t)s * TILE; };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int split = blockIdx.x, kvh = blockIdx.y;
    const DPlan plan(p, split);
    const float sl2 = (1.0f / sqrtf((float)D)) * kLog2e;

    // Launched with programmatic stream serialization.  When the kernel in front of us on the stream is the library's own
    // table kernel (bifocal), that kernel was launched normally, so everything the caller enqueued before the call --
    // the kernel that wrote q or appended KV row L-1 -- has completed before we run.  In the control (and G = 1) there is
    // no table kernel: wait for the predecessor here, before q or the cache are read (the prologue up to here still
    // overlaps its tail).
    if (!p.bifocal) griddep_wait();
    // the query loads go out before the TMA streams start: behind ~14 MB of in-flight cache tiles they take microseconds
    constexpr int NI = (NG * 64 + RT - 1) / RT;                        // (head, pair) items of the Q operands per rotate thread
    // rotate-group thread index.  Group warp w' = 2 (w & 3) + (w >> 2) for the CTA's rotate warp w = warp - 3: the odd w' (which
    // build the slow pairs' operand in SPLIT mode) and the even w' each land on all four sub-partitions
    const int rt = ((((warp - 3) & 3) * 2 + (((warp - 3) >> 2) & 1)) << 5) | lane;
    __nv_bfloat16 qv1[NI], qv2[NI];
    float2 tqh[NI], tql[NI];                       // HI / LO table entries of the query position
    KRot<RROWS> rot;
    bool tab_early = false;
    unsigned tab_gen = 0;                                               // check word of the table header at the early read
    const long long nq = (p.L - 1) - (p.L - 1) / p.G;                  // -Delta(q) >= 0, Eq.(5)
    // SPLIT: table entries of this thread's slow pair (rt & 63 >= 32): the unit step, the two possible steps of the reference
    // row from one tile to the next (n_ref advances by D0 or D0 + 1, D0 = 128 - ceil(128 / G)), the first tile's reference row
    float2 s_unit = make_float2(1.f, 0.f), s_e0 = s_unit, s_e1 = s_unit, s_rh = s_unit, s_rl = s_unit;
    const unsigned sD0 = 128u - (unsigned)((128 + p.G - 1) / p.G);
    auto load_tables = [&]() {
        if (p.split && (rt & 63) >= 32) {
            const int si = rt & 63;
            const unsigned pr = (unsigned)(plan.kt(0) * BN) + 64u, n = pr - pr / (unsigned)p.G;
            s_unit = __ldg(&p.lo[64 + si]);
            s_e0 = __ldg(&p.lo[(size_t)sD0 * 64 + si]);
            s_e1 = __ldg(&p.lo[(size_t)(sD0 + 1) * 64 + si]);
            s_rh = __ldg(&p.hi[(size_t)(n >> 8) * 64 + si]);
            s_rl = __ldg(&p.lo[(size_t)(n & 255) * 64 + si]);
        }
#pragma unroll
        for (int it = 0; it < NI; ++it) {
            const int idx = rt + it * RT;
            if (idx < p.g * 64) {
                tqh[it] = __ldg(&p.hi[(nq >> 8) * 64 + (idx & 63)]);
                tql[it] = __ldg(&p.lo[(nq & 255) * 64 + (idx & 63)]);
            }
        }
        // SPLIT: chunks 0-3 only.  The odd warps also build the slow pairs' operand every tile, so they rotate one row per
        // thread (rows 96-127) and the even warps three (rows 0-95): both halves of the group finish a tile together
        if (p.split) {
            const int e = (rt >> 6) * 8 + ((rt & 31) >> 2);
            
            rot.init_at(p.lo, p.hi, rt & 3, (rt & 32) ? 32 * (4 - RO) + RO * e : (4 - RO) * e, p.G);
        }
        else rot.init(p.lo, p.hi, rt, p.G);
        rot.seek((unsigned)(plan.kt(0) * BN));
        rot.prefetch_carried();
    };
    if (warp >= 3 && warp < 3 + RW) {
#pragma unroll
        for (int it = 0; it < NI; ++it) {
            const int idx = rt + it * RT;
            if (idx < p.g * 64) {
                const __nv_bfloat16* qh = p.q + (size_t)(kvh * p.gq + p.h0 + (idx >> 6)) * D;
                qv1[it] = qh[idx & 63];
                qv2[it] = qh[(idx & 63) + 64];
            }
        }
        // So do the table loads (Q' entries, the unit step, the first tile's first rows): once the streams run, an L2 hit
        // takes microseconds (measured: 8.4 k cycles from the first TMA to the first rotation, 1.7 k in the control).
        // The tables come from the preceding kernel, which rewrites them only when their header does not match (theta,
        // n_hi, d); if it matches NOW that kernel will find the same and write nothing, so they can be read before it ends.
        if (plan.nr > 0) {
            const volatile TableHeader* hdr =
                reinterpret_cast<const volatile TableHeader*>(reinterpret_cast<const unsigned char*>(p.lo) - 256);
            tab_early = hdr->magic == kTableMagic && hdr->theta == p.theta && hdr->n_hi == p.n_hi && hdr->d == D &&
                        hdr->interp == p.fm.interp &&
                        (!p.fm.interp || (hdr->omg == p.fm.one_minus_inv_G && hdr->w_pre == p.fm.w_pre && hdr->alpha == p.fm.alpha &&
                                          hdr->beta == p.fm.beta));
            tab_gen = hdr->check;                                     // the check word the header promises for the table body
            if (tab_early) load_tables();
            // verify the body ourselves, exactly as the table kernel does (hash of LO[1] and HI[n_hi-1], tables.cu): a CTA
            // whose check passes need not wait for that kernel at all
            if (rt < 128) {
                uint32_t h = 0;
                if (tab_early) {
                    const float2 v = rt < 64 ? p.lo[64 + rt] : p.hi[(p.n_hi - 1) * 64 + (rt - 64)];
                    h = (__float_as_uint(v.x) * 0x9E3779B1u) ^ (__float_as_uint(v.y) * 0x85EBCA77u) ^ ((uint32_t)rt * 0xC2B2AE3Du);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) h ^= __shfl_xor_sync(0xffffffffu, h, o);
                if (lane == 0) bars->chk[rt >> 5] = h;
            }
        }
    }
    griddep_launch_dependents();                                       // the merge kernel may queue up behind us
    if (tid == 0) {
        for (int i = 0; i < KS; ++i) { mbar_init(&bars->k_full[i], 1); mbar_init(&bars->k_ready[i], RW); mbar_init(&bars->k_empty[i], 1); }
        for (int i = 0; i < VS; ++i) { mbar_init(&bars->v_full[i], 1); mbar_init(&bars->v_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&bars->s_full[i], 1); mbar_init(&bars->p_full[i], 4); }
        mbar_init(&bars->pv_done, 1); mbar_init(&bars->o_full, 1); mbar_init(&bars->q_ready, RW);
        fence_barrier_init();
        prefetch_tmap(&tmK); prefetch_tmap(&tmV);
    }
    if (warp == 1) tmem_alloc<TM_COLS>(&bars->tmem_base);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bars->tmem_base;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            int pg_next = (pages && plan.nv > 0) ? __ldg(pages + plan.kt(0)) : 0;
            for (int v = 0; v < plan.nv; ++v) {
                const int row0 = (pages ? pg_next : plan.kt(v)) * BN;  // paged: physical page of the logical tile
                if (pages && v + 1 < plan.nv) pg_next = __ldg(pages + plan.kt(v + 1));   // in flight under the wait below
                const int s = v % KS;
                if (v >= KS) mbar_wait(&bars->k_empty[s], ((v / KS) - 1) & 1);
                mbar_arrive_expect_tx(&bars->k_full[s], TILE);
                tma_load_3d(sK(s), &tmK, &bars->k_full[s], 0, kvh, row0);
                tma_load_3d(sK(s) + BOXB, &tmK, &bars->k_full[s], 64, kvh, row0);
                if (PFK > 0 && p.bifocal && v + PFK < plan.nv) {                // tile v + 1 into L2: its load will be an L2 hit
                    const int row1 = (pages ? pg_next : plan.kt(v + PFK)) * BN;
                    tma_prefetch_3d(&tmK, 0, kvh, row1);
                    tma_prefetch_3d(&tmK, 64, kvh, row1);
                }
            }
        }
    } else if (warp == 2) {
        // ===================== TMA producer for V (its own thread: a V stage lives until O += V^T P of its visit,
        // much longer than a K stage, and must not hold back the K loads) =====================
        if (lane == 0) {
            int pg_next = (pages && plan.nv > 0) ? __ldg(pages + plan.kt(0)) : 0;
            for (int v = 0; v < plan.nv; ++v) {
                const int row0 = (pages ? pg_next : plan.kt(v)) * BN;
                if (pages && v + 1 < plan.nv) pg_next = __ldg(pages + plan.kt(v + 1));
                const int sv = v % VS;
                if (v >= VS) mbar_wait(&bars->v_empty[sv], ((v / VS) - 1) & 1);
                mbar_arrive_expect_tx(&bars->v_full[sv], TILE);
                tma_load_3d(sV(sv), &tmV, &bars->v_full[sv], 0, kvh, row0);
                tma_load_3d(sV(sv) + BOXB, &tmV, &bars->v_full[sv], 64, kvh, row0);
                if (PFV > 0 && p.bifocal && v + PFV < plan.nv) {
                    const int row1 = (pages ? pg_next : plan.kt(v + PFV)) * BN;
                    tma_prefetch_3d(&tmV, 0, kvh, row1);
                    tma_prefetch_3d(&tmV, 64, kvh, row1);
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (convergent warp, one elected lane issues) =====================
        const uint32_t tm = __shfl_sync(0xffffffffu, tmem, 0);
        const uint32_t smem0 = __shfl_sync(0xffffffffu, smem_u32(smem), 0);
        auto issue_s = [&](int v) {
            const uint32_t dS = tm + TM_S + (v & 1) * SCOLS;
            const uint32_t ka = smem0 + (v % KS) * KSTAGE, kla = ka + TILE;
            const uint32_t qa = smem0 + (uint32_t)OFF_Q;
            const bool rem = plan.remote(v);
            if (elect_one()) {
                if (!rem) {
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks)
                        umma_ss(dS, smem_desc_sw128(ka + (ks >> 2) * BOXB + (ks & 3) * 32, 16, 1024),
                                smem_desc_sw128(qa + (ks >> 2) * (NH * 128) + (ks & 3) * 32, 16, 1024), IDESC_S_BF16, ks > 0);
                } else if (p.split) {
                    const uint32_t qc = qa + QBUF;
                    // slow pairs first (they open columns 0-47): stored bf16 K slices 2, 3, 6, 7 times the per-tile operand
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int ks = (j & 1) + 2 + (j >> 1) * 4;
                        umma_ss(dS, smem_desc_sw128(ka + (ks >> 2) * BOXB + (ks & 3) * 32, 16, 1024),
                                smem_desc_sw128(kla + (j >> 1) * 64 * 128 + 32 + (j & 1) * 64, 16, 1024), IDESC_S_BF16_N48, j > 0);
                    }
#pragma unroll
                    for (int j = 0; j < 4; ++j) {              // fast pairs: K'hi [Q'hi ; Q'lo] on slices 0, 1, 4, 5 (columns 0-31)
                        const int ks = (j & 1) + (j >> 1) * 4;
                        umma_ss(dS, smem_desc_sw128(ka + (ks >> 2) * BOXB + (ks & 3) * 32, 16, 1024),
                                smem_desc_sw128(qc + (ks >> 2) * (2 * NH * 128) + (ks & 3) * 32, 16, 1024), IDESC_S_F16_N32, 1);
                    }
#pragma unroll
                    for (int ks = 0; ks < D / 32; ks += 2)     // K'lo (e5m2) Q'hi (e5m2) of channels 0-31 and 64-95
                        umma_ss_f8(dS, smem_desc_sw128(kla + ks * 32, 16, 1024),
                                   smem_desc_sw128(qc + QCBUF + ks * 32, 16, 1024), IDESC_S_E5M2 | (1u << 13), 1);
                } else {
                    const uint32_t qc = qa + QBUF;                  // rows 0-15 Q'hi, rows 16-31 Q'lo
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks)        // K'hi [Q'hi ; Q'lo]: one pass over the K tile, N = 32
                        umma_ss(dS, smem_desc_sw128(ka + (ks >> 2) * BOXB + (ks & 3) * 32, 16, 1024),
                                smem_desc_sw128(qc + (ks >> 2) * (2 * NH * 128) + (ks & 3) * 32, 16, 1024), IDESC_S_F16_N32, ks > 0);
#pragma unroll
                    for (int ks = 0; ks < D / 32; ++ks)        // K'lo (e5m2) Q'hi (e5m2) into columns 0-15
                        umma_ss_f8(dS, smem_desc_sw128(kla + ks * 32, 16, 1024),
                                   smem_desc_sw128(qc + QCBUF + ks * 32, 16, 1024), IDESC_S_E5M2 | (1u << 13), 1);   // K' lo is stored negated (rotate_rows2): negate A
                }
                umma_commit(&bars->s_full[v & 1]);
                umma_commit(&bars->k_empty[v % KS]);
            }
            __syncwarp();
        };
        auto issue_pv = [&](int v) {
            const uint32_t va = smem0 + (uint32_t)OFF_V + (v % VS) * TILE;
            const uint32_t pa = smem0 + (uint32_t)OFF_P;
            if (elect_one()) {
#pragma unroll
                for (int ks = 0; ks < BN / 16; ++ks)
                    umma_ss(tm + TM_O, smem_desc_sw128(va + ks * 2048, BOXB, 1024),
                            smem_desc_sw128(pa + (ks >> 2) * (NH * 128) + (ks & 3) * 32, 16, 1024), IDESC_PV,
                            (v > 0 || ks > 0) ? 1u : 0u);
                umma_commit(&bars->v_empty[v % VS]);
                umma_commit(&bars->pv_done);
            }
            __syncwarp();
        };
        mbar_wait(&bars->q_ready, 0);
        for (int v = 0; v <= plan.nv; ++v) {
            if (v < plan.nv) {
                mbar_wait(&bars->k_ready[v % KS], (v / KS) & 1);
                tc_fence_after();
                issue_s(v);
            }
            if (v > 0) {
                const int u = v - 1;
                mbar_wait(&bars->p_full[u & 1], (u >> 1) & 1);
                mbar_wait(&bars->v_full[u % VS], (u / VS) & 1);
                tc_fence_after();
                issue_pv(u);
            }
        }
        if (elect_one()) umma_commit(&bars->o_full);
        __syncwarp();
    } else if (warp >= 3 && warp < 3 + RW) {
        // ===================== rotate group (steps a4, a5) =====================
        const int t = rt;
        // Q operands [16 heads][128 ch]: raw bf16 for local tiles; Q' = R(Delta q) Q as fp16 hi / lo for remote tiles
        for (int i = t; i < (QBUF + QCBUF + QYBUF) / 4; i += RT) reinterpret_cast<uint32_t*>(sQ)[i] = 0u;
        for (int i = t; i < QBUF / 4; i += RT) reinterpret_cast<uint32_t*>(sP)[i] = 0u;
        named_bar_sync(1, RT);
        if (plan.nr > 0) {
            // header sealed for these parameters AND the body verified against its check word (partial hashes of rotate
            // warps 0-3, exchanged by the named barrier above): the early loads stand.  Otherwise the table kernel is
            // rebuilding (or about to): wait for it, then load.
            const uint32_t mine = (bars->chk[0] ^ bars->chk[1] ^ bars->chk[2] ^ bars->chk[3]) | 1u;
            if (!tab_early || mine != tab_gen) {
                griddep_wait();
                load_tables();
            }
        }
        float qy1[NI], qy2[NI];                 // Q' pairs of this thread in fp32 (SPLIT: the slow ones are re-based per tile)
#pragma unroll
        for (int it = 0; it < NI; ++it) { qy1[it] = 0.f; qy2[it] = 0.f; }
#pragma unroll
        for (int it = 0; it < NI; ++it) {                  // (no break: the register arrays keep static indices)
            const int idx = t + it * RT;
            const bool mine = idx < p.g * 64;
            const int h = idx >> 6, i = idx & 63;
            const __nv_bfloat16 b1 = qv1[it], b2 = qv2[it];
            if (mine) {
                *reinterpret_cast<__nv_bfloat16*>(sQ + bop_off(h, i)) = b1;
                *reinterpret_cast<__nv_bfloat16*>(sQ + bop_off(h, i + 64)) = b2;
            }
            if (mine && plan.nr > 0) {
                const float2 ch = tqh[it], cl = tql[it];
                const float c = ch.x * cl.x - ch.y * cl.y, s = ch.y * cl.x + ch.x * cl.y;
                const float x1 = __bfloat162float(b1), x2 = __bfloat162float(b2);
                const float y1 = x1 * c - x2 * s, y2 = x1 * s + x2 * c;
                qy1[it] = y1; qy2[it] = y2;
                const __half h1 = __float2half_rn(y1), h2 = __float2half_rn(y2);
                *reinterpret_cast<__half*>(sQ + QBUF + bop_off<2 * NH>(h, i)) = h1;
                *reinterpret_cast<__half*>(sQ + QBUF + bop_off<2 * NH>(h, i + 64)) = h2;
                *reinterpret_cast<__half*>(sQ + QBUF + bop_off<2 * NH>(NH + h, i)) = __float2half_rn(y1 - __half2float(h1));
                *reinterpret_cast<__half*>(sQ + QBUF + bop_off<2 * NH>(NH + h, i + 64)) = __float2half_rn(y2 - __half2float(h2));
                // Q'hi as e5m2 (top byte of the fp16, rounded): byte ch of row h, 16-byte chunks swizzled by (h & 7)
                unsigned char* qy = sQ + QBUF + QCBUF + h * 128;
                qy[(((i >> 4) ^ (h & 7)) << 4) + (i & 15)] = (unsigned char)((__half_as_ushort(h1) + 0x80) >> 8);
                qy[((((i + 64) >> 4) ^ (h & 7)) << 4) + (i & 15)] = (unsigned char)((__half_as_ushort(h2) + 0x80) >> 8);
            }
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->q_ready);
        // SPLIT: this thread's slow pair i = t & 63 (>= 32) of heads (t >> 6) + 4 it; table entries of the tile's reference row
        const int si = t & 63;
        const bool slow = p.split && plan.nr > 0 && si >= 32;
        // sin of the unit step = its angle a_i to 2e-7 (|a_i| <= 1.1e-3); -a_i^2 / 2; cs(alpha_ref) of the current tile, carried
        // from tile to tile by one complex multiplication (no table load inside the loop: an L2 hit behind the cache
        // streams takes longer than a tile)
        const float ua = s_unit.y, ub = -0.5f * ua * ua;
        float rc = s_rh.x * s_rl.x - s_rh.y * s_rl.y, rs = s_rh.y * s_rl.x + s_rh.x * s_rl.y;
        // n_ref advances by 128 - floor(128 / G) - [phase wraps], phase = (reference position) mod G: no division per tile
        const unsigned gG = (unsigned)p.G, g_m = 128u % gG, g_d = 128u / gG;
        unsigned g_ph = ((unsigned)(plan.kt(0) * BN) + 64u) % gG;
        const uint32_t sb0 = (uint32_t)((si < 48 ? 32 : 96) + (si & 15) * 2);     // byte of channel i in its operand row
        for (int v = 0; v < plan.nv; ++v) {
            const int s = v % KS;
            if (slow && plan.remote(v)) {
                // The slow pairs' operand of tile v does not depend on the tile: it is written while the tile is still in flight.
                // Its bytes are free once the MMAs of the stage's previous tile have completed (k_empty, the barrier the K
                // producer waited on before it issued this tile's load).
                const uint32_t kl = smem_u32(sK(s)) + TILE;
                if (v >= KS) mbar_wait(&bars->k_empty[s], ((v / KS) - 1) & 1);
                const float c = rc, sn = rs;                                 // cs(alpha_ref) of pair i
                {
                    g_ph += g_m;
                    const bool wrap = g_ph >= gG;                            // one more multiple of G passed: n_ref advances by D0
                    if (wrap) g_ph -= gG;
                    const float2 e = (wrap || g_m == 0u) ? s_e0 : s_e1;
                    rc = c * e.x - sn * e.y; rs = sn * e.x + c * e.y;
                }
#pragma unroll
                for (int it = 0; it < NI; ++it) {
                    const int h = (t >> 6) + 4 * it;
                    if (h < p.g) {
                        const float q1 = c * qy1[it] + sn * qy2[it], q2 = c * qy2[it] - sn * qy1[it];   // qt = Rot(alpha_ref)^T q'
                        const uint16_t h1 = bf16_bits(q1), h2 = bf16_bits(q2);
                        const float r1 = q1 - __uint_as_float((uint32_t)h1 << 16), r2 = q2 - __uint_as_float((uint32_t)h2 << 16);
                        const float u1 = ua * q2, u2 = -ua * q1;                     // a J^T qt: hi and lo as well -- its bf16
                        const uint16_t g1 = bf16_bits(u1), g2 = bf16_bits(u2);       // rounding alone is 64 theta_i 2^-9 of a full-size term
                        const float v1 = u1 - __uint_as_float((uint32_t)g1 << 16), v2 = u2 - __uint_as_float((uint32_t)g2 << 16);
                        // blocks 0, 2, 3, 4, 5: column 16 + h is where the fast pairs put their Q'lo term, which like qt lo
                        // is not multiplied by dn; block 1 (columns 8-15) is never written and never read
                        const uint16_t w1[5] = {h1, bf16_bits(r1), g1, bf16_bits(v1), bf16_bits(ub * q1)};     // channel i
                        const uint16_t w2[5] = {h2, bf16_bits(r2), g2, bf16_bits(v2), bf16_bits(ub * q2)};     // channel i + 64
                        // row 8 b + h of the operand: the swizzle term depends on h only (8 rows = one swizzle period)
                        const uint32_t a = kl + (uint32_t)h * 128 + ((((sb0 >> 4) ^ ((uint32_t)h & 7u)) << 4) | (sb0 & 15u));
#pragma unroll
                        for (int b = 0; b < 5; ++b) {
                            const int blk = b == 0 ? 0 : b + 1;
                            sts16(a + blk * SB * 128, w1[b]);
                            sts16(a + blk * SB * 128 + 64 * 128, w2[b]);
                        }
                    }
                }
            }
            mbar_wait(&bars->k_full[s], (v / KS) & 1);
            if (plan.remote(v) && p.split) {
                const uint32_t kl = smem_u32(sK(s)) + TILE;
                if (t & 32) rotate_rows2<RO, BOXB, 3, true, true>(smem_u32(sK(s)), kl, (unsigned)(plan.kt(v) * BN), rot, SelTree(), 0u, 0u);
                else rotate_rows2<4 - RO, BOXB, 3, true, true>(smem_u32(sK(s)), kl, (unsigned)(plan.kt(v) * BN), rot, SelTree(), 0u, 0u);
                fence_proxy_async_smem();
                if (plan.remote(v + 1)) { rot.step128(g_m, g_d); rot.prefetch_carried(); }
            } else if (plan.remote(v)) {
                rotate_rows2<RROWS, BOXB, 3, true, true>(smem_u32(sK(s)), smem_u32(sK(s)) + TILE, (unsigned)(plan.kt(v) * BN), rot, SelTree(), 0u, 0u);
                fence_proxy_async_smem();
                if (plan.remote(v + 1)) { rot.step128(g_m, g_d); rot.prefetch_carried(); }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars->k_ready[s]);
        }
    } else {
        // ===================== softmax group (steps a6-a8): one thread per key of the tile =====================
        const int wq = warp & 3;                                     // TMEM lane quadrant of this warp
        const int j = (wq << 5) | lane;                              // key row in the tile == TMEM lane
        const uint32_t lane_base = (uint32_t)(wq << 5) << 16;
        const int g = p.g;
        const uint32_t pb = smem_u32(sP) + (j >> 6) * (NH * 128) + (j & 7) * 2;   // P[h][j] = pb + h*128 + ((cj ^ (h&7)) << 4)
        const int cj = (j & 63) >> 3;
        float m_ref[NG], l[NG];
#pragma unroll
        for (int h = 0; h < NG; ++h) { m_ref[h] = -INFINITY; l[h] = 0.f; }
        for (int v = 0; v < plan.nv; ++v) {
            const long long key = (long long)plan.kt(v) * BN + j;
            const bool valid = plan.remote(v) ? (key >= plan.ks && key < plan.re) : (key >= plan.ls && key < plan.ke);
            float dn = 0.f;                                           // SPLIT: n(key) - n(reference row), ahead of the wait for S
            if (p.split && plan.remote(v)) {
                const unsigned pk = (unsigned)key, pr = (unsigned)(plan.kt(v) * BN) + 64u, Gu = (unsigned)p.G;
                dn = (float)((int)(pk - pk / Gu) - (int)(pr - pr / Gu));
            }
            mbar_wait(&bars->s_full[v & 1], (v >> 1) & 1);
            tc_fence_after();
            uint32_t sr[32];
            tmem_ld32(tmem + lane_base + TM_S + (v & 1) * SCOLS, sr);
            const bool rem = plan.remote(v);                          // remote: columns 16.. hold the K'hi Q'lo term
            float tay[NG];                                            // SPLIT: dn (S[.,2] + dn S[.,3]) of the slow pairs
#pragma unroll
            for (int h = 0; h < NG; ++h) tay[h] = 0.f;
            if (rem && p.split) {
                uint32_t st[16];                                       // columns 32-47: a J^T qt lo | -a^2/2 qt
                tmem_ld16(tmem + lane_base + TM_S + (v & 1) * SCOLS + 2 * NH, st);
                tmem_ld_wait();
#pragma unroll
                for (int h = 0; h < NG && h < SB; ++h)
                    tay[h] = dn * ((__uint_as_float(sr[3 * SB + h]) + __uint_as_float(st[h])) + dn * __uint_as_float(st[SB + h]));
            } else {
                tmem_ld_wait();
            }
            float x[NG];
            bool jump = false;
#pragma unroll
            for (int h = 0; h < NG; ++h) {
                const float sc = __uint_as_float(sr[h]) + (rem ? __uint_as_float(sr[NH + h]) + tay[h] : 0.0f);
                x[h] = (valid && h < g) ? sc * sl2 : -INFINITY;
                jump |= x[h] > m_ref[h] + 8.0f;                      // lazy rescale: only on a jump of 2^8 (or from -inf)
            }
            if (bar_red_or(2, 128, jump)) {                          // rare; uniform over the 128 threads
                float tmax[NG];
#pragma unroll
                for (int h = 0; h < NG; ++h) {
                    float w = x[h];
#pragma unroll
                    for (int off = 16; off >= 1; off >>= 1) w = fmaxf(w, __shfl_xor_sync(0xffffffffu, w, off));
                    tmax[h] = w;
                }
                if (lane < NG) {
                    float w = -INFINITY;
#pragma unroll
                    for (int h = 0; h < NG; ++h) if (lane == h) w = tmax[h];
                    bars->red[wq * NH + lane] = w;
                }
                named_bar_sync(2, 128);
                float alpha[NG];
#pragma unroll
                for (int h = 0; h < NG; ++h) {
                    const float* red = bars->red;
                    const float tm_h = fmaxf(fmaxf(red[h], red[NH + h]), fmaxf(red[2 * NH + h], red[3 * NH + h]));
                    alpha[h] = 1.0f;
                    if (tm_h > m_ref[h]) {
                        alpha[h] = (m_ref[h] == -INFINITY) ? 0.0f : ex2(m_ref[h] - tm_h);
                        m_ref[h] = tm_h;
                        l[h] *= alpha[h];
                    }
                }
                named_bar_sync(2, 128);                              // red[] may be rewritten by the next slow path
                if (v > 0) {                                         // O^T row of channel j: scale column h by alpha[h]
                    mbar_wait(&bars->pv_done, (v - 1) & 1);
                    tc_fence_after();
                    uint32_t og[16];
                    tmem_ld16(tmem + lane_base + TM_O, og);
                    tmem_ld_wait();
#pragma unroll
                    for (int h = 0; h < NG; ++h) og[h] = __float_as_uint(__uint_as_float(og[h]) * alpha[h]);
                    tmem_st16(tmem + lane_base + TM_O, og);
                    tmem_st_wait();
                    tc_fence_before();
                }
            }
            if (v > 0) mbar_wait(&bars->pv_done, (v - 1) & 1);        // single P buffer: O += V^T P of visit v-1 has read it
#pragma unroll
            for (int h = 0; h < NG; ++h) {
                const float pr = (x[h] == -INFINITY) ? 0.0f : ex2(x[h] - m_ref[h]);
                l[h] += pr;
                if (h < g) sts16(pb + h * 128 + ((cj ^ (h & 7)) << 4), bf16_bits(pr));
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars->p_full[v & 1]);
        }
        // ---- partial state of this split (steps a7, a8): l summed over the 128 key lanes, O^T from TMEM ----------
#pragma unroll
        for (int h = 0; h < NG; ++h) {
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) l[h] += __shfl_xor_sync(0xffffffffu, l[h], off);
        }
        if (lane < NG) {
            float w = 0.f;
#pragma unroll
            for (int h = 0; h < NG; ++h) if (lane == h) w = l[h];
            bars->red[wq * NH + lane] = w;
        }
        named_bar_sync(2, 128);
        mbar_wait(&bars->o_full, 0);
        tc_fence_after();
        uint32_t og[16];
        if (plan.nv > 0) {
            tmem_ld16(tmem + lane_base + TM_O, og);
            tmem_ld_wait();
        } else {
#pragma unroll
            for (int h = 0; h < 16; ++h) og[h] = 0u;
        }
        constexpr int SS = D + 2;
        griddep_wait();                                              // the previous step's merge may still be reading the partials
#pragma unroll
        for (int h = 0; h < NG; ++h) {
            if (h < g) {
                float* dst = p.part + ((size_t)split * p.H_q + (size_t)kvh * p.gq + p.h0 + h) * SS;
                dst[j] = __uint_as_float(og[h]);
                if (j == 0) {
                    dst[D] = m_ref[h];
                    dst[D + 1] = bars->red[h] + bars->red[NH + h] + bars->red[2 * NH + h] + bars->red[3 * NH + h];
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<TM_COLS>(tmem);
}

}  // namespace

// SPLIT holds when the in-tile phase of pair 32 stays small: 64 theta_32 = 64 rope_theta^-1/2 <= 0.095, i.e. rope_theta >= 4.54e5
// (third-order term of the rotation <= 1.4e-4 per pair; Llama-3's 5e5 is inside).  Measured on the stress input with loud pairs
// 32 / 33 at rope_theta = 5e5 / 4.2e5 / 4.1e5: lse error 2.5e-4 / 3.2e-4 / 5.6e-4 with SPLIT against 8.1e-4 / 9.5e-4 / - with the
// per-key rotation (fp16 + e5m2 residual of a loud pair): the bound is set by the expansion's own error, with a factor 2 in hand.  The frequency-interpolation map keeps the per-key rotation.
static int split_ok(double theta, const FreqMap& fm, int g) {
    return (!fm.interp && g <= SB && 64.0 / sqrt(theta) <= 0.095) ? 1 : 0;
}

bool umma_decode_supported(int H_q, int H_kv, int d, int dtype) {
    return dtype == JETLONG_BF16 && d == 128 && H_kv >= 1 && H_q % H_kv == 0;     // any group size: 16 heads per launch
}
bool umma_decode_paged_supported(int H_q, int H_kv, int d, int dtype) {
    return umma_decode_supported(H_q, H_kv, d, dtype) && H_q / H_kv <= NH;
}

// split plan: one CTA per SM (the kernel needs ~215 KB of shared memory), key ranges are multiples of the 128-key tile
void umma_decode_plan(long long L, int H_kv, int* nsplit, long long* kps) {
    const long long ntiles = (L + BN - 1) / BN;
    long long ns = sm_count() / H_kv;
    if (ns < 1) ns = 1;
    if (ns > ntiles) ns = ntiles;
    if (ns > 1024) ns = 1024;
    const long long tps = (ntiles + ns - 1) / ns;
    *kps = tps * BN;
    *nsplit = (int)((ntiles + tps - 1) / tps);
}

int launch_decode_umma(const void* q, const void* K, const void* V, float* part, long long L, int H_q, int H_kv,
                       long long w0, long long G, double theta, bool bifocal, const float2* lo, const float2* hi,
                       int* nsplit_out, cudaStream_t st, FreqMap fm) {
    CUtensorMap tmK, tmV;
    if (!make_kv_tensor_map(&tmK, K, L, H_kv, BN) || !make_kv_tensor_map(&tmV, V, L, H_kv, BN)) return JETLONG_UNSUPPORTED;
    Params p;
    p.q = (const __nv_bfloat16*)q;
    p.part = part;
    p.L = L; p.w0 = w0; p.G = G;
    int ns;
    umma_decode_plan(L, H_kv, &ns, &p.kps);
    p.H_q = H_q; p.H_kv = H_kv; p.gq = H_q / H_kv;
    p.bifocal = bifocal ? 1 : 0;
    p.lo = lo; p.hi = hi;
    p.theta = theta;
    p.n_hi = (L + 255) / 256 + 1; p.fm = fm;
    BatchInfo bi = {};                                                 // batch = 0: the single-sequence call
    // More than 16 query heads per KV head: one launch per 16 heads of the group (the head operand is N = 16), each streaming
    // the cache again; the launches write disjoint partials and chain by programmatic serialization (each waits for its
    // predecessor before it writes, so the merge behind the last one sees them all).
    for (int h0 = 0; h0 < p.gq; h0 += NH) {
        p.h0 = h0;
        p.g = p.gq - h0 < NH ? p.gq - h0 : NH;
        p.split = bifocal ? split_ok(theta, fm, p.g) : 0;
        auto kern = p.g <= 1 ? decode_umma_kernel<1, false> : p.g <= 2 ? decode_umma_kernel<2, false> : p.g <= 4 ? decode_umma_kernel<4, false>
                  : p.g <= 8 ? decode_umma_kernel<8, false> : decode_umma_kernel<16, false>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess)
            return check_launch("decode_umma attr");
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(ns, H_kv);
        cfg.blockDim = dim3(NTHREADS);
        cfg.dynamicSmemBytes = SMEM_BYTES;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, kern, tmK, tmV, p, bi);
        note_launch();
    }
    *nsplit_out = ns;
    return check_launch("decode_umma_kernel");
}

// Batched decode over a paged cache: up to MAXB sequences per launch (grid z), each with its own length / group size.
// Kpool, Vpool: [pool_pages * 128, H_kv, 128]; the split count follows the longest sequence.
int launch_decode_umma_paged(const void* q, const void* Kpool, const void* Vpool, const int* page_table, int max_pages,
                             long long pool_pages, const long long* Ls, const long long* Gs, int nb, float* part,
                             long long part_stride, long long Lmax, int H_q, int H_kv, long long w0, double theta,
                             const float2* lo, const float2* hi, int* nsplit_out, cudaStream_t st) {
    CUtensorMap tmK, tmV;
    if (!make_kv_tensor_map(&tmK, Kpool, pool_pages * BN, H_kv, BN) || !make_kv_tensor_map(&tmV, Vpool, pool_pages * BN, H_kv, BN))
        return JETLONG_UNSUPPORTED;
    if (nb < 1 || nb > MAXB) return JETLONG_INVALID_ARG;
    Params p;
    p.q = (const __nv_bfloat16*)q;
    p.part = part;
    p.L = Lmax; p.w0 = w0; p.G = 1;
    int ns;
    umma_decode_plan(Lmax, H_kv * nb, &ns, &p.kps);                    // one CTA per SM over all (sequence, KV head) pairs
    p.H_q = H_q; p.H_kv = H_kv; p.g = H_q / H_kv; p.gq = p.g; p.h0 = 0;
    p.bifocal = 0;
    p.lo = lo; p.hi = hi;
    p.theta = theta;
    p.n_hi = (Lmax + 255) / 256 + 1; p.fm = alias_map();
    p.split = split_ok(theta, p.fm, p.g);
    BatchInfo bi = {};
    bi.batch = nb; bi.page_table = page_table; bi.max_pages = max_pages; bi.part_stride = part_stride;
    bool any_bifocal = false;
    for (int b = 0; b < MAXB; ++b) {
        bi.Ls[b] = b < nb ? Ls[b] : 1;
        bi.Gs[b] = b < nb ? (int)Gs[b] : 1;
        if (b < nb && Gs[b] > 1 && w0 < Ls[b] - 1) any_bifocal = true;
    }
    auto kern = p.g <= 1 ? decode_umma_kernel<1, true> : p.g <= 2 ? decode_umma_kernel<2, true> : p.g <= 4 ? decode_umma_kernel<4, true>
              : p.g <= 8 ? decode_umma_kernel<8, true> : decode_umma_kernel<16, true>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess)
        return check_launch("decode_umma attr");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ns, H_kv, nb);
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = any_bifocal ? 1 : 0;                                // without the table kernel in front: a normal launch
    cudaLaunchKernelEx(&cfg, kern, tmK, tmV, p, bi);
    note_launch();
    *nsplit_out = ns;
    return check_launch("decode_umma_kernel (paged)");
}

}  // namespace jetlong
