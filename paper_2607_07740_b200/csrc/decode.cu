// decode.cu -- split-KV batch-1 bifocal / causal decode (step a9, merge a7, epilogue a8).
//
// One query row per head at position L-1 against cache rows 0..L-1.  Keys with
// k >= L-1-w0 are local (stored q, stored k); older keys are corrected in registers,
// k' = R(Delta k) k (Eq.(5)-(6) P:101-106); the cache is only ever read.
//
// HBM-bound scan: grid = (splits, ceil(H_kv/HPB), g/GQ).  A CTA owns a contiguous key range; warp w
// owns one KV head, so the (cos, sin) of Delta(k) -- which do not depend on the head -- are built once
// per 64-key chunk in shared memory and shared by all heads of the CTA.  Each lane loads 16 bytes of a
// K row and 16 bytes of the V row (128-bit coalesced), the GQ query heads of the group share them.
// Partial (m, l, O) states go to the workspace and are merged by decode_merge_kernel (additive LSE
// merge, Eq.(7) without the minus sign).
#include <math.h>

#include "common.cuh"

namespace jetlong {

namespace {

constexpr int NW = 8;              // warps per CTA
constexpr int CK = 64;             // keys per cs chunk
constexpr float kLog2e = 1.4426950408889634f;

template <typename T> struct Lane;
template <> struct Lane<__nv_bfloat16> {
    static constexpr int EPL = 8;
    static __device__ inline void unpack(const uint4& u, float* f) {
        f[0] = __uint_as_float(u.x << 16); f[1] = __uint_as_float(u.x & 0xffff0000u);
        f[2] = __uint_as_float(u.y << 16); f[3] = __uint_as_float(u.y & 0xffff0000u);
        f[4] = __uint_as_float(u.z << 16); f[5] = __uint_as_float(u.z & 0xffff0000u);
        f[6] = __uint_as_float(u.w << 16); f[7] = __uint_as_float(u.w & 0xffff0000u);
    }
};
template <> struct Lane<float> {
    static constexpr int EPL = 4;
    static __device__ inline void unpack(const uint4& u, float* f) {
        f[0] = __uint_as_float(u.x); f[1] = __uint_as_float(u.y);
        f[2] = __uint_as_float(u.z); f[3] = __uint_as_float(u.w);
    }
};

__device__ inline uint4 ldg_stream(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

struct DecodeParams {
    const void* q; const void* K; const void* V;
    float* part;                    // [nsplit][H_q][D+2]
    long long L, w0, G, kps;        // kps = keys per split (multiple of CK)
    int H_q, H_kv, HPB;             // HPB = KV heads per CTA (1,2,4,8)
    const float2* lo; const float2* hi;
};

// two-level lookup: (cos, sin)(Delta theta_i), Delta <= 0
__device__ inline float2 cs_lookup(const float2* __restrict__ lo, const float2* __restrict__ hi, long long delta,
                                   int half, int i) {
    const long long n = -delta;
    const float2 h = __ldg(&hi[(n >> 8) * half + i]);
    const float2 l = __ldg(&lo[(n & 255) * half + i]);
    return make_float2(h.x * l.x - h.y * l.y, h.y * l.x + h.x * l.y);
}

template <typename T, int D, int GQ, bool BIFOCAL>
__global__ void __launch_bounds__(NW * 32) decode_kernel(DecodeParams p) {
    constexpr int EPL = Lane<T>::EPL;
    constexpr int LPR = D / EPL;                 // lanes per row
    constexpr int RPW = 32 / LPR;                // rows per warp iteration
    constexpr int HL = LPR / 2;                  // lanes per half row
    constexpr int HALF = D / 2;
    constexpr int PIECES = EPL / 2;              // 16-byte pieces of cs per lane per key
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* cs_buf = reinterpret_cast<float2*>(smem_raw);        // [2][CK][HALF] (permuted rows)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int sub = lane % LPR, rsel = lane / LPR;
    const bool second = sub >= HL;
    const int fchunk = sub % HL;
    const int WPH = NW / p.HPB;                  // warps per KV head
    const int kvh = blockIdx.y * p.HPB + (warp % p.HPB);
    const int wsub = warp / p.HPB;
    const bool active = kvh < p.H_kv;
    const int g = p.H_q / p.H_kv;
    const int hq0 = kvh * g + blockIdx.z * GQ;   // first query head of this warp
    const long long qpos = p.L - 1;
    const long long kb = (BIFOCAL && qpos - p.w0 > 0) ? qpos - p.w0 : 0;   // keys >= kb are local
    const long long ks = (long long)blockIdx.x * p.kps;
    const long long ke = (ks + p.kps < p.L) ? ks + p.kps : p.L;
    const float sl2 = (1.0f / sqrtf((float)D)) * kLog2e;

    // ---- this lane's slice of the GQ query rows: stored q and q' = R(Delta q) q (step a4) -------------
    float ql[GQ][EPL], qr[GQ][EPL];
    if (active) {
        float csq_c[EPL], csq_s[EPL];
#pragma unroll
        for (int e = 0; e < EPL; ++e) {
            float2 cs = make_float2(1.f, 0.f);
            if (BIFOCAL) cs = cs_lookup(p.lo, p.hi, delta_pos(qpos, p.G), HALF, fchunk * EPL + e);
            csq_c[e] = cs.x;
            csq_s[e] = second ? cs.y : -cs.y;
        }
#pragma unroll
        for (int h = 0; h < GQ; ++h) {
            const uint4 u = *reinterpret_cast<const uint4*>(reinterpret_cast<const T*>(p.q) +
                                                            (size_t)(hq0 + h) * D + sub * EPL);
            Lane<T>::unpack(u, ql[h]);
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                const float other = __shfl_xor_sync(0xffffffffu, ql[h][e], HL);
                qr[h][e] = (ql[h][e] * csq_c[e] + other * csq_s[e]) * sl2;
            }
#pragma unroll
            for (int e = 0; e < EPL; ++e) ql[h][e] *= sl2;      // scores come out in log2 units
        }
    }
    float m[GQ], l[GQ], o[GQ][EPL];
#pragma unroll
    for (int h = 0; h < GQ; ++h) {
        m[h] = -INFINITY; l[h] = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) o[h][e] = 0.f;
    }

    auto process_row = [&](const uint4& ku, const uint4& vu, const float (*qq)[EPL], const float2* csrow,
                           bool rotate) {
        float kf[EPL], vf[EPL];
        Lane<T>::unpack(ku, kf);
        if (rotate) {
            float c[EPL], s[EPL];
#pragma unroll
            for (int pc = 0; pc < PIECES; ++pc) {
                const float4 t = *reinterpret_cast<const float4*>(&csrow[(pc * HL + fchunk) * 2]);
                c[2 * pc] = t.x; s[2 * pc] = t.y; c[2 * pc + 1] = t.z; s[2 * pc + 1] = t.w;
            }
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                const float other = __shfl_xor_sync(0xffffffffu, kf[e], HL);
                kf[e] = kf[e] * c[e] + other * (second ? s[e] : -s[e]);
            }
        }
        float sc[GQ];
#pragma unroll
        for (int h = 0; h < GQ; ++h) {
            float a = 0.f;
#pragma unroll
            for (int e = 0; e < EPL; ++e) a = fmaf(qq[h][e], kf[e], a);
            sc[h] = a;
        }
#pragma unroll
        for (int off = LPR / 2; off >= 1; off >>= 1)
#pragma unroll
            for (int h = 0; h < GQ; ++h) sc[h] += __shfl_xor_sync(0xffffffffu, sc[h], off);
        Lane<T>::unpack(vu, vf);
#pragma unroll
        for (int h = 0; h < GQ; ++h) {
            if (sc[h] > m[h]) {                                   // lazy rescale: rare after warm-up
                const float a = exp2f(m[h] - sc[h]);              // m = -inf -> 0
                l[h] *= a;
#pragma unroll
                for (int e = 0; e < EPL; ++e) o[h][e] *= a;
                m[h] = sc[h];
            }
            const float pr = exp2f(sc[h] - m[h]);
            l[h] += pr;
#pragma unroll
            for (int e = 0; e < EPL; ++e) o[h][e] = fmaf(pr, vf[e], o[h][e]);
        }
    };

    const T* Kp = reinterpret_cast<const T*>(p.K);
    const T* Vp = reinterpret_cast<const T*>(p.V);
    const size_t row_stride = (size_t)p.H_kv * D;
    const size_t lane_off = (size_t)kvh * D + sub * EPL;

    // ---- remote phase: keys [ks, min(ke, kb)) --------------------------------------------------------
    if (BIFOCAL) {
        const long long re = ke < kb ? ke : kb;
        int buf = 0;
        for (long long c0 = ks; c0 < re; c0 += CK, buf ^= 1) {
            float2* csb = cs_buf + (size_t)buf * CK * HALF;
            for (int idx = tid; idx < CK * HALF; idx += NW * 32) {          // step a5 coefficients
                const int j = idx / HALF, i = idx - j * HALF;
                const long long k = c0 + j;
                float2 cs = make_float2(1.f, 0.f);
                if (k < re) cs = cs_lookup(p.lo, p.hi, delta_pos(k, p.G), HALF, i);
                const int cch = i / EPL, e = i % EPL;
                csb[(size_t)j * HALF + ((e >> 1) * HL + cch) * 2 + (e & 1)] = cs;
            }
            __syncthreads();      // chunk ready; also fences reuse of the other buffer (double-buffered)
            if (active) {
                constexpr int UN = 4;
                const int step = WPH * RPW;
                for (int j0 = wsub * RPW + rsel; j0 < CK; j0 += step * UN) {
                    uint4 ku[UN], vu[UN];
#pragma unroll
                    for (int u = 0; u < UN; ++u) {
                        const int j = j0 + u * step;
                        const long long k = c0 + j;
                        if (j < CK && k < re) {
                            ku[u] = ldg_stream(Kp + (size_t)k * row_stride + lane_off);
                            vu[u] = ldg_stream(Vp + (size_t)k * row_stride + lane_off);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < UN; ++u) {
                        const int j = j0 + u * step;
                        // all lanes of a row group share j; groups may diverge at the tail, shuffles stay
                        // inside the LPR-lane group, so run under a group-uniform predicate mask-free.
                        const bool ok = (j < CK) && (c0 + j < re);
                        if (__all_sync(0xffffffffu, ok)) {
                            process_row(ku[u], vu[u], qr, csb + (size_t)j * HALF, true);
                        } else if (__any_sync(0xffffffffu, ok)) {
                            // ragged tail: every lane executes the shuffles, only valid groups commit
                            const int jj = ok ? j : 0;
                            float m_s[GQ], l_s[GQ], o_s[GQ][EPL];
#pragma unroll
                            for (int h = 0; h < GQ; ++h) {
                                m_s[h] = m[h]; l_s[h] = l[h];
#pragma unroll
                                for (int e = 0; e < EPL; ++e) o_s[h][e] = o[h][e];
                            }
                            uint4 kz = ok ? ku[u] : make_uint4(0, 0, 0, 0), vz = ok ? vu[u] : make_uint4(0, 0, 0, 0);
                            process_row(kz, vz, qr, csb + (size_t)jj * HALF, true);
                            if (!ok) {
#pragma unroll
                                for (int h = 0; h < GQ; ++h) {
                                    m[h] = m_s[h]; l[h] = l_s[h];
#pragma unroll
                                    for (int e = 0; e < EPL; ++e) o[h][e] = o_s[h][e];
                                }
                            }
                        }
                    }
                }
            }
        }
    }
    // ---- local phase: keys [max(ks, kb), ke) -- stored q, stored k, no rotation --------------------------
    if (active) {
        constexpr int UN = 4;
        const long long ls = ks > kb ? ks : kb;
        const long long step = (long long)WPH * RPW;
        for (long long k0 = ls + wsub * RPW + rsel; k0 - rsel - wsub * RPW < ke; k0 += step * UN) {
            uint4 ku[UN], vu[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const long long k = k0 + u * step;
                if (k < ke) {
                    ku[u] = ldg_stream(Kp + (size_t)k * row_stride + lane_off);
                    vu[u] = ldg_stream(Vp + (size_t)k * row_stride + lane_off);
                }
            }
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const bool ok = (k0 + u * step) < ke;
                if (__all_sync(0xffffffffu, ok)) {
                    process_row(ku[u], vu[u], ql, nullptr, false);
                } else if (__any_sync(0xffffffffu, ok)) {
                    float m_s[GQ], l_s[GQ], o_s[GQ][EPL];
#pragma unroll
                    for (int h = 0; h < GQ; ++h) {
                        m_s[h] = m[h]; l_s[h] = l[h];
#pragma unroll
                        for (int e = 0; e < EPL; ++e) o_s[h][e] = o[h][e];
                    }
                    uint4 kz = ok ? ku[u] : make_uint4(0, 0, 0, 0), vz = ok ? vu[u] : make_uint4(0, 0, 0, 0);
                    process_row(kz, vz, ql, nullptr, false);
                    if (!ok) {
#pragma unroll
                        for (int h = 0; h < GQ; ++h) {
                            m[h] = m_s[h]; l[h] = l_s[h];
#pragma unroll
                            for (int e = 0; e < EPL; ++e) o[h][e] = o_s[h][e];
                        }
                    }
                }
            }
        }
    }

    // ---- merge the CTA's (warp, row-group) states, write one partial per query head (step a7) ----------
    __syncthreads();
    float* st = reinterpret_cast<float*>(smem_raw);               // [NW][RPW][GQ][D+2]
    constexpr int SS = D + 2;
    {
        float* mine = st + (((size_t)warp * RPW + rsel) * GQ) * SS;
#pragma unroll
        for (int h = 0; h < GQ; ++h) {
#pragma unroll
            for (int e = 0; e < EPL; ++e) mine[h * SS + sub * EPL + e] = active ? o[h][e] : 0.f;
            if (sub == 0) { mine[h * SS + D] = active ? m[h] : -INFINITY; mine[h * SS + D + 1] = active ? l[h] : 0.f; }
        }
    }
    __syncthreads();
    const int heads_cta = p.HPB * GQ;
    for (int idx = tid; idx < heads_cta * SS; idx += NW * 32) {
        const int hh = idx / SS, e = idx - hh * SS;
        const int hp = hh / GQ, h = hh - hp * GQ;                 // KV head slot in CTA, query head in group
        const int kvh2 = blockIdx.y * p.HPB + hp;
        if (kvh2 >= p.H_kv) continue;
        float M = -INFINITY;
        for (int ws = 0; ws < WPH; ++ws)
            for (int r = 0; r < RPW; ++r)
                M = fmaxf(M, st[(((size_t)(ws * p.HPB + hp) * RPW + r) * GQ + h) * SS + D]);
        float acc = 0.f;
        if (M != -INFINITY) {
            for (int ws = 0; ws < WPH; ++ws)
                for (int r = 0; r < RPW; ++r) {
                    const float* s = st + (((size_t)(ws * p.HPB + hp) * RPW + r) * GQ + h) * SS;
                    const float w = exp2f(s[D] - M);
                    if (e < D) acc += w * s[e];
                    else if (e == D + 1) acc += w * s[D + 1];
                }
        }
        const int hq = kvh2 * g + blockIdx.z * GQ + h;
        p.part[((size_t)blockIdx.x * p.H_q + hq) * SS + e] = (e == D) ? M : acc;
    }
}

// ---- split merge: warp-shuffle log-sum-exp over the splits (step a7 (ii), a8) ---------------------------
template <typename T, int D>
__global__ void __launch_bounds__(D) decode_merge_kernel(const float* __restrict__ part, int nsplit, int H_q,
                                                         T* __restrict__ out, float* __restrict__ lse,
                                                         long long part_stride = 0) {
    constexpr int SS = D + 2;
    part += (size_t)blockIdx.y * part_stride;                       // batched decode: grid y = sequence
    out += (size_t)blockIdx.y * H_q * D;
    lse += (size_t)blockIdx.y * H_q;
    __shared__ float w_s[1024];
    __shared__ float red[2];
    const int h = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    asm volatile("griddepcontrol.wait;" ::: "memory");           // launched programmatically behind the scan kernel
    if (tid < 32) {
        float M = -INFINITY;
        for (int s = lane; s < nsplit; s += 32) M = fmaxf(M, part[((size_t)s * H_q + h) * SS + D]);
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, off));
        float lsum = 0.f;
        for (int s = lane; s < nsplit; s += 32) {
            const float* ps = part + ((size_t)s * H_q + h) * SS;
            const float w = exp2f(ps[D] - M);                      // empty split: m = -inf -> w = 0
            w_s[s] = w;
            lsum += w * ps[D + 1];
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, off);
        if (lane == 0) { red[0] = M; red[1] = lsum; }
    }
    __syncthreads();
    float acc = 0.f;
    for (int s = 0; s < nsplit; ++s) acc += w_s[s] * part[((size_t)s * H_q + h) * SS + tid];
    out[(size_t)h * D + tid] = from_f32<T>(acc / red[1]);
    if (tid == 0) lse[h] = (red[0] + log2f(red[1])) * 0.6931471805599453f;   // back to natural log
}

struct Plan { int nsplit; long long kps; int HPB; int GQ; int gz; int gy; };

Plan make_plan(long long L, int H_q, int H_kv) {
    Plan pl;
    pl.HPB = H_kv >= 8 ? 8 : (H_kv >= 4 ? 4 : (H_kv >= 2 ? 2 : 1));
    pl.gy = (H_kv + pl.HPB - 1) / pl.HPB;
    const int g = H_q / H_kv;
    pl.GQ = (g % 4 == 0) ? 4 : ((g % 2 == 0) ? 2 : 1);
    pl.gz = g / pl.GQ;
    const int target = sm_count() * 2;
    int ns = target / (pl.gy * pl.gz);
    if (ns < 1) ns = 1;
    if (ns > 1024) ns = 1024;
    long long kps = (L + ns - 1) / ns;
    kps = ((kps + CK - 1) / CK) * CK;
    pl.kps = kps;
    pl.nsplit = (int)((L + kps - 1) / kps);
    return pl;
}

}  // namespace

// decode_umma.cu
bool umma_decode_supported(int H_q, int H_kv, int d, int dtype);
void umma_decode_plan(long long L, int H_kv, int* nsplit, long long* kps);
int launch_decode_umma(const void* q, const void* K, const void* V, float* part, long long L, int H_q, int H_kv,
                       long long w0, long long G, double theta, bool bifocal, const float2* lo, const float2* hi,
                       int* nsplit_out, cudaStream_t st, FreqMap fm);

size_t decode_workspace_bytes(long long L, int H_q, int H_kv, int d) {
    // room for the partials of either implementation (SIMT or tcgen05) at this L
    Plan pl = make_plan(L, H_q, H_kv);
    int ns = pl.nsplit, nu = 0;
    long long kps = 0;
    umma_decode_plan(L, H_kv, &nu, &kps);
    if (nu > ns) ns = nu;
    return two_level_bytes(L, d) + align256((size_t)ns * H_q * (d + 2) * sizeof(float));
}

template <typename T, int D>
static int launch_decode_td(const void* q, const void* K, const void* V, void* out, float* lse, long long L,
                            int H_q, int H_kv, long long w0, long long G, double theta, bool bifocal, void* ws,
                            cudaStream_t st, FreqMap fm) {
    Plan pl = make_plan(L, H_q, H_kv);
    unsigned char* base = (unsigned char*)ws;
    const size_t tb = two_level_bytes(L, D);
    if (bifocal) {
        int rc = build_two_level(base, L, D, theta, st, fm);
        if (rc != JETLONG_OK) return rc;
    }
    DecodeParams p;
    p.q = q; p.K = K; p.V = V;
    p.part = reinterpret_cast<float*>(base + tb);
    p.L = L; p.w0 = w0; p.G = G; p.kps = pl.kps;
    p.H_q = H_q; p.H_kv = H_kv; p.HPB = pl.HPB;
    p.lo = reinterpret_cast<const float2*>(base + 256);
    p.hi = p.lo + 256 * (D / 2);
    if (umma_decode_supported(H_q, H_kv, D, sizeof(T) == 2 ? JETLONG_BF16 : JETLONG_FP32)) {
        int ns = 0;
        int rc = launch_decode_umma(q, K, V, p.part, L, H_q, H_kv, w0, G, theta, bifocal, p.lo, p.hi, &ns, st, fm);
        if (rc != JETLONG_OK) return rc;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(H_q);
        cfg.blockDim = dim3(D);
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, decode_merge_kernel<T, D>, (const float*)p.part, ns, H_q, (T*)out, lse, 0ll);
        note_launch();
        return check_launch("decode_merge_kernel");
    }
    const size_t cs_bytes = 2 * (size_t)CK * (D / 2) * sizeof(float2);
    constexpr int EPL = Lane<T>::EPL;
    const size_t st_bytes = (size_t)NW * (32 / (D / EPL)) * 4 * (D + 2) * sizeof(float);
    const size_t smem = cs_bytes > st_bytes ? cs_bytes : st_bytes;
    dim3 grid(pl.nsplit, pl.gy, pl.gz);
#define JL_DEC(GQv)                                                                                          \
    {                                                                                                        \
        auto kern = bifocal ? decode_kernel<T, D, GQv, true> : decode_kernel<T, D, GQv, false>;              \
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                  \
        kern<<<grid, NW * 32, smem, st>>>(p);                                                                \
    }
    if (pl.GQ == 4) JL_DEC(4) else if (pl.GQ == 2) JL_DEC(2) else JL_DEC(1)
#undef JL_DEC
    note_launch();
    int rc = check_launch("decode_kernel");
    if (rc != JETLONG_OK) return rc;
    decode_merge_kernel<T, D><<<H_q, D, 0, st>>>(p.part, pl.nsplit, H_q, (T*)out, lse);
    note_launch();
    return check_launch("decode_merge_kernel");
}

int launch_decode_umma_paged(const void* q, const void* Kpool, const void* Vpool, const int* page_table, int max_pages,
                             long long pool_pages, const long long* Ls, const long long* Gs, int nb, float* part,
                             long long part_stride, long long Lmax, int H_q, int H_kv, long long w0, double theta,
                             const float2* lo, const float2* hi, int* nsplit_out, cudaStream_t st);

size_t decode_paged_workspace_bytes(long long Lmax, int batch, int H_q, int H_kv, int d) {
    int ns = 0;
    long long kps = 0;
    umma_decode_plan(Lmax, H_kv, &ns, &kps);                         // an upper bound of the splits of any launch
    return two_level_bytes(Lmax, d) + (size_t)batch * align256((size_t)ns * H_q * (d + 2) * sizeof(float));
}

// batch > 1 over a paged cache (bf16, d = 128, tcgen05 path): chunks of up to 16 sequences per launch
int launch_decode_paged(const void* q, const void* Kpool, const void* Vpool, const int* page_table, int max_pages,
                        long long pool_pages, const long long* Ls, const long long* Gs, int batch, void* out, float* lse,
                        int H_q, int H_kv, long long w0, double theta, void* ws, cudaStream_t st) {
    constexpr int D = 128;
    long long Lmax = 1;
    bool any_bifocal = false;
    for (int b = 0; b < batch; ++b) {
        if (Ls[b] > Lmax) Lmax = Ls[b];
        if (Gs[b] > 1 && w0 < Ls[b] - 1) any_bifocal = true;
    }
    unsigned char* base = (unsigned char*)ws;
    const size_t tb = two_level_bytes(Lmax, D);
    if (any_bifocal) {
        int rc = build_two_level(base, Lmax, D, theta, st);          // the table does not depend on G: one for every sequence
        if (rc != JETLONG_OK) return rc;
    }
    const float2* lo = reinterpret_cast<const float2*>(base + 256);
    const float2* hi = lo + 256 * (D / 2);
    int ns0 = 0;
    long long kps0 = 0;
    umma_decode_plan(Lmax, H_kv, &ns0, &kps0);
    const long long part_stride = (long long)(align256((size_t)ns0 * H_q * (D + 2) * sizeof(float)) / sizeof(float));
    float* part = reinterpret_cast<float*>(base + tb);
    for (int b0 = 0; b0 < batch; b0 += 16) {
        const int nb = batch - b0 < 16 ? batch - b0 : 16;
        int ns = 0;
        int rc = launch_decode_umma_paged((const __nv_bfloat16*)q + (size_t)b0 * H_q * D, Kpool, Vpool,
                                          page_table + (size_t)b0 * max_pages, max_pages, pool_pages, Ls + b0, Gs + b0, nb,
                                          part + (size_t)b0 * part_stride, part_stride, Lmax, H_q, H_kv, w0, theta, lo, hi, &ns, st);
        if (rc != JETLONG_OK) return rc;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(H_q, nb);
        cfg.blockDim = dim3(D);
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, decode_merge_kernel<__nv_bfloat16, D>, (const float*)(part + (size_t)b0 * part_stride), ns, H_q,
                           (__nv_bfloat16*)out + (size_t)b0 * H_q * D, lse + (size_t)b0 * H_q, part_stride);
        note_launch();
        rc = check_launch("decode_merge_kernel (paged)");
        if (rc != JETLONG_OK) return rc;
    }
    return JETLONG_OK;
}

int launch_decode(const void* q, const void* K, const void* V, void* out, float* lse, long long L, int H_q, int H_kv,
                  int d, long long w0, long long G, double theta, int dtype, bool bifocal, void* ws, size_t ws_bytes,
                  cudaStream_t st, FreqMap fm) {
    (void)ws_bytes;
    if (dtype == JETLONG_FP32) {
        if (d == 64) return launch_decode_td<float, 64>(q, K, V, out, lse, L, H_q, H_kv, w0, G, theta, bifocal, ws, st, fm);
        return launch_decode_td<float, 128>(q, K, V, out, lse, L, H_q, H_kv, w0, G, theta, bifocal, ws, st, fm);
    }
    if (d == 64)
        return launch_decode_td<__nv_bfloat16, 64>(q, K, V, out, lse, L, H_q, H_kv, w0, G, theta, bifocal, ws, st, fm);
    return launch_decode_td<__nv_bfloat16, 128>(q, K, V, out, lse, L, H_q, H_kv, w0, G, theta, bifocal, ws, st, fm);
}

}  // namespace jetlong
