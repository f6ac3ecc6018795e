// prefill_umma.cu -- tcgen05 UMMA bifocal / causal prefill for bf16, head_dim 128 (steps a3-a8, a10).
//
// One CTA = 128 query rows x 2 query heads of one KV group ("tile A", "tile B"): both see the same keys,
// the same positions and therefore the same tile classification, so one TMA-loaded K tile, one V tile and
// one in-smem RoPE correction (Eq.(6)) serve both.  Warp roles (512 threads):
//   warp 0      TMA producer: Q (once), then one K and one V tile per visit, SWIZZLE_128B boxes
//   warp 1      MMA issuer: S_t = Q_t K^T (tcgen05.mma SS), O_t += P_t V (tcgen05.mma TS, P from TMEM)
//   warps 4-7   rotate group: remote visits rotate the K tile in shared memory between the TMA load and the
//               MMA (bf16 -> fp32 rotate -> fp16, in place); once per CTA it turns Q into Q' = R(Delta q) Q
//   warps 8-11  softmax group of tile A; warps 12-15 softmax group of tile B (one thread per query row)
// TMEM (512 columns): S_A | S_B | O_A | O_B, 128 fp32 columns each; P_t (bf16) aliases S_t columns 0..63.
//
// Visit order per CTA: local visits first (diagonal tile, then the band down to q - w0), then the Q -> Q'
// switch, then the remote visits.  The straddle tile is visited twice with complementary masks (step a6).
// All visits feed ONE running (m, l, O) per row: the additive form of the Eq.(7) merge.
//
// Precision: local visits multiply the stored bf16 Q, K.  Remote operands are rounded once to fp16
// (kind::f16 takes fp16 as well as bf16; values are far inside the fp16 range), see DESIGN.md.
#include <cuda.h>
#include <math.h>

#include "common.cuh"
#include "umma.cuh"

namespace jetlong {

namespace {

using namespace ptx;

constexpr int D = 128, BM = 128, BN = 128;
constexpr int KS = 3, VS = 2;                         // K / V ring depths
constexpr int TILE_BYTES = BM * D * 2;                // 32 KB: two 16 KB SWIZZLE_128B boxes (cols 0-63 | 64-127)
constexpr int BOX_BYTES = 128 * 128;
constexpr int NTHREADS = 512;
constexpr float kLog2e = 1.4426950408889634f;

struct Bars {
    uint64_t q_full, q_local_done, q_rot_done, o_full;
    uint64_t k_full[KS], k_ready[KS], k_empty[KS];
    uint64_t v_full[VS], v_empty[VS];
    uint64_t s_full[2], p_full[2];
    uint32_t tmem_base;
};

constexpr size_t SMEM_BYTES = 1024 /*align slack*/ + (size_t)(2 + KS + VS) * TILE_BYTES + 1024 /*Bars*/;

struct Params {
    __nv_bfloat16* out;
    float* lse;
    long long L, w0, G;
    int H_q, H_kv, g;
    int bifocal;
    const float2* lo;
    const float2* hi;
};

struct Visit { int kt; int mode; };                   // mode 0 = causal/control, 1 = local, 2 = remote

struct Plan {
    int qb, n_local, n_remote, kt_hi, nv;
    __device__ Plan(int qb_, long long w0, bool bifocal) : qb(qb_) {
        const long long q0 = (long long)qb * BM;
        if (!bifocal) { n_local = qb + 1; n_remote = 0; kt_hi = -1; nv = n_local; return; }
        long long t = q0 - w0 - (BN - 1);                              // local iff k0 >= t
        long long kt_lo = t <= 0 ? 0 : (t + BN - 1) / BN;
        n_local = (int)(qb - kt_lo + 1);
        long long u = q0 + (BM - 1) - 1 - w0;                          // remote iff k0 <= u  (q0+127-k0 > w0)
        kt_hi = u < 0 ? -1 : (int)(u / BN);
        if (kt_hi > qb) kt_hi = qb;
        n_remote = kt_hi + 1;
        nv = n_local + n_remote;
    }
    __device__ Visit at(int v, bool bifocal) const {
        Visit x;
        if (v < n_local) { x.kt = qb - v; x.mode = bifocal ? 1 : 0; }
        else { x.kt = kt_hi - (v - n_local); x.mode = 2; }
        return x;
    }
};

// ---- step a4 / a5: in-place correction rotation of a [128 rows][128 ch] SWIZZLE_128B tile, bf16 -> fp16 ----
// Row r of the tile sits at absolute position pos0 + r.  Thread t of the 128-thread rotate group owns the
// 16-byte chunk c = t & 7 (channels 8c..8c+7 of box 0 and their partners 64+8c.. of box 1) of rows 8(t>>3)+m.
__device__ __forceinline__ void rotate_tile(unsigned char* tile, long long pos0, long long G,
                                            const float2* __restrict__ lo, const float2* __restrict__ hi, int t) {
    const int c = t & 7;
#pragma unroll 2
    for (int m = 0; m < 8; ++m) {
        const int r = 8 * (t >> 3) + m;
        const long long pos = pos0 + r;
        const long long n = pos - pos / G;                              // -Delta(pos) >= 0, Eq.(5)
        const float4* ph = reinterpret_cast<const float4*>(hi + (n >> 8) * 64 + 8 * c);
        const float4* pl = reinterpret_cast<const float4*>(lo + (n & 255) * 64 + 8 * c);
        float cs_c[8], cs_s[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float4 h = __ldg(ph + j), l = __ldg(pl + j);
            cs_c[2 * j] = h.x * l.x - h.y * l.y;      cs_s[2 * j] = h.y * l.x + h.x * l.y;
            cs_c[2 * j + 1] = h.z * l.z - h.w * l.w;  cs_s[2 * j + 1] = h.w * l.z + h.z * l.w;
        }
        unsigned char* p1 = tile + r * 128 + ((c ^ (r & 7)) << 4);
        unsigned char* p2 = p1 + BOX_BYTES;
        const uint4 u1 = *reinterpret_cast<const uint4*>(p1);
        const uint4 u2 = *reinterpret_cast<const uint4*>(p2);
        const uint32_t a[4] = {u1.x, u1.y, u1.z, u1.w}, b[4] = {u2.x, u2.y, u2.z, u2.w};
        uint32_t o1[4], o2[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float x1l = __uint_as_float(a[j] << 16), x1h = __uint_as_float(a[j] & 0xffff0000u);
            const float x2l = __uint_as_float(b[j] << 16), x2h = __uint_as_float(b[j] & 0xffff0000u);
            const float y1l = x1l * cs_c[2 * j] - x2l * cs_s[2 * j];
            const float y2l = x1l * cs_s[2 * j] + x2l * cs_c[2 * j];
            const float y1h = x1h * cs_c[2 * j + 1] - x2h * cs_s[2 * j + 1];
            const float y2h = x1h * cs_s[2 * j + 1] + x2h * cs_c[2 * j + 1];
            __half2 h1 = __floats2half2_rn(y1l, y1h), h2 = __floats2half2_rn(y2l, y2h);
            o1[j] = *reinterpret_cast<uint32_t*>(&h1);
            o2[j] = *reinterpret_cast<uint32_t*>(&h2);
        }
        *reinterpret_cast<uint4*>(p1) = make_uint4(o1[0], o1[1], o1[2], o1[3]);
        *reinterpret_cast<uint4*>(p2) = make_uint4(o2[0], o2[1], o2[2], o2[3]);
    }
}

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

constexpr uint32_t IDESC_QK_BF16 = idesc_f16(1, 1, 0, 0, BM, BN);
constexpr uint32_t IDESC_QK_F16 = idesc_f16(0, 0, 0, 0, BM, BN);
constexpr uint32_t IDESC_PV = idesc_f16(1, 1, 0, 1, BM, D);      // A = P (TMEM, bf16), B = V (smem, MN-major)

__global__ void __launch_bounds__(NTHREADS, 1)
prefill_umma_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                    const __grid_constant__ CUtensorMap tmV, const Params p) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    unsigned char* sQ = smem;
    unsigned char* sK = sQ + 2 * TILE_BYTES;
    unsigned char* sV = sK + KS * TILE_BYTES;
    Bars* bars = reinterpret_cast<Bars*>(sV + VS * TILE_BYTES);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_qb = (int)((p.L + BM - 1) / BM);
    const int pairs = p.H_q / 2;
    const int qb = n_qb - 1 - (int)(blockIdx.x / pairs);          // heaviest row blocks first
    const int h0 = 2 * (int)(blockIdx.x % pairs);
    const int kvh = h0 / p.g;
    const long long q0 = (long long)qb * BM;
    const bool bifocal = p.bifocal != 0;
    const Plan plan(qb, p.w0, bifocal);

    if (tid == 0) {
        mbar_init(&bars->q_full, 1); mbar_init(&bars->q_local_done, 1); mbar_init(&bars->q_rot_done, 128);
        mbar_init(&bars->o_full, 1);
        for (int i = 0; i < KS; ++i) { mbar_init(&bars->k_full[i], 1); mbar_init(&bars->k_ready[i], 128); mbar_init(&bars->k_empty[i], 1); }
        for (int i = 0; i < VS; ++i) { mbar_init(&bars->v_full[i], 1); mbar_init(&bars->v_empty[i], 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(&bars->s_full[i], 1); mbar_init(&bars->p_full[i], 128); }
        fence_barrier_init();
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV);
    }
    if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bars->tmem_base;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            mbar_arrive_expect_tx(&bars->q_full, 2 * TILE_BYTES);
            for (int t = 0; t < 2; ++t)
                for (int b = 0; b < 2; ++b)
                    tma_load_3d(sQ + t * TILE_BYTES + b * BOX_BYTES, &tmQ, &bars->q_full, 64 * b, h0 + t, (int)q0);
            for (int v = 0; v < plan.nv; ++v) {
                const Visit x = plan.at(v, bifocal);
                const int s = v % KS, sv = v % VS;
                if (v >= KS) mbar_wait(&bars->k_empty[s], ((v / KS) - 1) & 1);
                mbar_arrive_expect_tx(&bars->k_full[s], TILE_BYTES);
                for (int b = 0; b < 2; ++b)
                    tma_load_3d(sK + s * TILE_BYTES + b * BOX_BYTES, &tmK, &bars->k_full[s], 64 * b, kvh, x.kt * BN);
                if (v >= VS) mbar_wait(&bars->v_empty[sv], ((v / VS) - 1) & 1);
                mbar_arrive_expect_tx(&bars->v_full[sv], TILE_BYTES);
                for (int b = 0; b < 2; ++b)
                    tma_load_3d(sV + sv * TILE_BYTES + b * BOX_BYTES, &tmV, &bars->v_full[sv], 64 * b, kvh, x.kt * BN);
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (one thread) =====================
        if (lane == 0) {
            auto issue_qk = [&](int v, int t) {
                const Visit x = plan.at(v, bifocal);
                const uint32_t idesc = x.mode == 2 ? IDESC_QK_F16 : IDESC_QK_BF16;
                const uint32_t a0 = smem_u32(sQ + t * TILE_BYTES), b0 = smem_u32(sK + (v % KS) * TILE_BYTES);
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t off = (ks >> 2) * BOX_BYTES + (ks & 3) * 32;
                    umma_ss(tmem + t * 128, smem_desc_sw128(a0 + off, 16, 1024), smem_desc_sw128(b0 + off, 16, 1024),
                            idesc, ks > 0);
                }
                umma_commit(&bars->s_full[t]);
            };
            auto issue_pv = [&](int v, int t) {
                const uint32_t b0 = smem_u32(sV + (v % VS) * TILE_BYTES);
#pragma unroll
                for (int ks = 0; ks < BN / 16; ++ks)
                    umma_ts(tmem + 256 + t * 128, tmem + t * 128 + ks * 8,
                            smem_desc_sw128(b0 + ks * 2048, BOX_BYTES, 1024), IDESC_PV, (v > 0 || ks > 0) ? 1u : 0u);
            };
            mbar_wait(&bars->q_full, 0);
            mbar_wait(&bars->k_ready[0], 0);
            tc_fence_after();
            issue_qk(0, 0);
            issue_qk(0, 1);
            umma_commit(&bars->k_empty[0]);
            if (plan.n_remote > 0 && plan.n_local == 1) umma_commit(&bars->q_local_done);
            for (int v = 0; v < plan.nv; ++v) {
                const int sv = v % VS;
                for (int t = 0; t < 2; ++t) {
                    mbar_wait(&bars->p_full[t], v & 1);
                    if (t == 0) mbar_wait(&bars->v_full[sv], (v / VS) & 1);
                    tc_fence_after();
                    issue_pv(v, t);
                    if (t == 1) umma_commit(&bars->v_empty[sv]);
                    if (v + 1 < plan.nv) {
                        if (t == 0) {
                            if (v + 1 == plan.n_local) mbar_wait(&bars->q_rot_done, 0);
                            mbar_wait(&bars->k_ready[(v + 1) % KS], ((v + 1) / KS) & 1);
                            tc_fence_after();
                        }
                        issue_qk(v + 1, t);
                        if (t == 1) {
                            umma_commit(&bars->k_empty[(v + 1) % KS]);
                            if (plan.n_remote > 0 && v + 1 == plan.n_local - 1) umma_commit(&bars->q_local_done);
                        }
                    }
                }
            }
            umma_commit(&bars->o_full);
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== rotate group (steps a4, a5) =====================
        const int t = tid - 128;
        for (int v = 0; v < plan.nv; ++v) {
            const Visit x = plan.at(v, bifocal);
            const int s = v % KS;
            mbar_wait(&bars->k_full[s], (v / KS) & 1);
            if (x.mode == 2) {
                if (v == plan.n_local) {                              // first remote visit: Q -> Q' = R(Delta q) Q
                    mbar_wait(&bars->q_local_done, 0);
                    rotate_tile(sQ, q0, p.G, p.lo, p.hi, t);
                    rotate_tile(sQ + TILE_BYTES, q0, p.G, p.lo, p.hi, t);
                    fence_proxy_async_smem();
                    mbar_arrive(&bars->q_rot_done);
                }
                rotate_tile(sK + s * TILE_BYTES, (long long)x.kt * BN, p.G, p.lo, p.hi, t);
                fence_proxy_async_smem();
            }
            mbar_arrive(&bars->k_ready[s]);
        }
    } else if (warp >= 8) {
        // ===================== softmax groups (steps a6-a8): one thread per query row =====================
        const int t = (warp - 8) >> 2;
        const int r = ((warp & 3) << 5) | lane;
        const uint32_t lane_base = (uint32_t)((warp & 3) << 5) << 16;
        const uint32_t tS = tmem + lane_base + t * 128, tO = tmem + lane_base + 256 + t * 128;
        const float sl2 = (1.0f / sqrtf((float)D)) * kLog2e;
        float m_ref = -INFINITY, l = 0.f;
        for (int v = 0; v < plan.nv; ++v) {
            const Visit x = plan.at(v, bifocal);
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
            mbar_wait(&bars->s_full[t], v & 1);
            tc_fence_after();
            uint32_t rg[32];
            float mx = -INFINITY;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
                tmem_ld32(tS + ch * 32, rg);
                tmem_ld_wait();
                if (masked) {
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const int c = ch * 32 + j;
                        mx = fmaxf(mx, (c >= lo && c <= hi) ? __uint_as_float(rg[j]) : -INFINITY);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j) mx = fmaxf(mx, __uint_as_float(rg[j]));
                }
            }
            const float mnew = mx * sl2;
            if (v == 0) {
                m_ref = mnew;
            } else {
                const bool need = mnew > m_ref + 8.0f;                 // lazy rescale: only on a jump of 2^8
                if (__any_sync(0xffffffffu, need)) {
                    const float alpha = need ? ex2(m_ref - mnew) : 1.0f;
                    if (need) m_ref = mnew;
                    l *= alpha;
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) {
                        tmem_ld32(tO + ch * 32, rg);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 32; ++j) rg[j] = __float_as_uint(__uint_as_float(rg[j]) * alpha);
                        tmem_st32(tO + ch * 32, rg);
                    }
                }
            }
            float sum = 0.f;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
                tmem_ld32(tS + ch * 32, rg);
                tmem_ld_wait();
                uint32_t pk[16];
#pragma unroll
                for (int j = 0; j < 32; j += 2) {
                    const int c = ch * 32 + j;
                    float a = ex2(fmaf(__uint_as_float(rg[j]), sl2, -m_ref));
                    float b = ex2(fmaf(__uint_as_float(rg[j + 1]), sl2, -m_ref));
                    if (masked) {
                        if (c < lo || c > hi) a = 0.f;
                        if (c + 1 < lo || c + 1 > hi) b = 0.f;
                    }
                    sum += a + b;
                    __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
                    pk[j >> 1] = *reinterpret_cast<uint32_t*>(&h);
                }
                tmem_st16(tS + ch * 16, pk);
            }
            l += sum;
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(&bars->p_full[t]);
        }
        // ---- epilogue (step a8) ----
        mbar_wait(&bars->o_full, 0);
        tc_fence_after();
        const long long q = q0 + r;
        const float inv = 1.0f / l;
        __nv_bfloat16* orow = p.out + ((size_t)q * p.H_q + (h0 + t)) * D;
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
            uint32_t rg[32];
            tmem_ld32(tO + ch * 32, rg);
            tmem_ld_wait();
            if (q < p.L) {
#pragma unroll
                for (int j = 0; j < 32; j += 8) {
                    uint32_t w[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        __nv_bfloat162 h = __floats2bfloat162_rn(__uint_as_float(rg[j + 2 * e]) * inv,
                                                                 __uint_as_float(rg[j + 2 * e + 1]) * inv);
                        w[e] = *reinterpret_cast<uint32_t*>(&h);
                    }
                    *reinterpret_cast<uint4*>(orow + ch * 32 + j) = make_uint4(w[0], w[1], w[2], w[3]);
                }
            }
        }
        if (q < p.L) p.lse[(size_t)(h0 + t) * p.L + q] = (m_ref + log2f(l)) * 0.6931471805599453f;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem);
}

// ---- host side ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
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

// [L, H, 128] bf16 tensor seen as (d, H, L); box = 64 channels x 1 head x 128 rows, SWIZZLE_128B, OOB rows -> 0
bool make_map(CUtensorMap* m, const void* base, long long L, int H) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)H, (cuuint64_t)L};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)H * D * 2};
    cuuint32_t box[3] = {64, 1, 128};
    cuuint32_t es[3] = {1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool umma_prefill_supported(long long L, int H_q, int H_kv, int d, int dtype) {
    if (dtype != JETLONG_BF16 || d != 128 || H_kv < 1 || H_q % H_kv) return false;
    const int g = H_q / H_kv;
    return (g % 2) == 0 && L >= 1 && L < (1ll << 30);
}

size_t umma_prefill_workspace_bytes(long long L, int, int, int d) { return two_level_bytes(L + 256, d); }

int launch_prefill_umma(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                        int H_kv, int d, long long w0, long long G, double theta, bool bifocal, void* ws,
                        size_t ws_bytes, cudaStream_t st) {
    (void)ws_bytes;
    CUtensorMap tmQ, tmK, tmV;
    if (!make_map(&tmQ, Q, L, H_q) || !make_map(&tmK, K, L, H_kv) || !make_map(&tmV, V, L, H_kv))
        return JETLONG_UNSUPPORTED;
    Params p;
    p.out = (__nv_bfloat16*)out;
    p.lse = lse;
    p.L = L; p.w0 = w0; p.G = G;
    p.H_q = H_q; p.H_kv = H_kv; p.g = H_q / H_kv;
    p.bifocal = bifocal ? 1 : 0;
    p.lo = nullptr; p.hi = nullptr;
    if (bifocal) {
        int rc = build_two_level(ws, L + 256, d, theta, st);
        if (rc != JETLONG_OK) return rc;
        p.lo = reinterpret_cast<const float2*>((unsigned char*)ws + 256);
        p.hi = p.lo + 256 * (d / 2);
    }
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(prefill_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) !=
            cudaSuccess)
            return check_launch("prefill_umma attr");
        attr_set = true;
    }
    const int n_qb = (int)((L + BM - 1) / BM);
    const unsigned grid = (unsigned)n_qb * (unsigned)(H_q / 2);
    prefill_umma_kernel<<<grid, NTHREADS, SMEM_BYTES, st>>>(tmQ, tmK, tmV, p);
    note_launch();
    return check_launch("prefill_umma_kernel");
}

}  // namespace jetlong
