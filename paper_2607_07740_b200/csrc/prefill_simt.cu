// prefill_simt.cu -- fp32-FMA tiled bifocal / causal prefill (steps a3-a8, a10 of the scope table).
//
// This is the exact-arithmetic path: fp32 inputs (config 1; tolerances 1e-4 / 1e-5 rule out tensor
// cores) and the bring-up / cross-check path for bf16 inputs.  One CTA = 64 query rows of one head;
// it walks 64-key tiles, classifies each (skip / local / remote / straddle, Eq.(1)), rotates
// the K tile in shared memory for the remote visit (Eq.(6)) and keeps ONE online-softmax
// state (m, l, O) per row, i.e. the additive form of the Eq.(7) merge.
#include <math.h>

#include "common.cuh"

namespace jetlong {

namespace {

constexpr int BM = 64, BN = 64, NT = 128;

template <int D> struct Smem {
    static constexpr int LD = D + 4;                 // padded row stride (floats): conflict-free LDS.128
    float q[BM * LD];                                // stored (local) queries
    float qr[BM * LD];                               // R(Delta q) Q  (remote queries)
    float k[BN * LD];
    float v[BN * D];
    float s[BM * (BN + 1)];
    float m[BM], l[BM], alpha[BM];
};

// S[r][c] = scale * <A[r], K[c]> for this thread's 4x8 micro-tile, masked, written to sm.s
template <int D>
__device__ inline void qk_tile(Smem<D>& sm, const float* __restrict__ A, int tid, float scale, long long q0,
                               long long k0, long long w0, int visit /*0 causal,1 local,2 remote*/) {
    constexpr int LD = Smem<D>::LD;
    const int ty = tid >> 3, tx = tid & 7;            // rows ty+16i, cols tx+8j
    float acc[4][8];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
#pragma unroll 4
    for (int kk = 0; kk < D; kk += 4) {
        float4 a[4], b[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = *reinterpret_cast<const float4*>(&A[(ty + 16 * i) * LD + kk]);
#pragma unroll
        for (int j = 0; j < 8; ++j) b[j] = *reinterpret_cast<const float4*>(&sm.k[(tx + 8 * j) * LD + kk]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                acc[i][j] = fmaf(a[i].x, b[j].x, acc[i][j]);
                acc[i][j] = fmaf(a[i].y, b[j].y, acc[i][j]);
                acc[i][j] = fmaf(a[i].z, b[j].z, acc[i][j]);
                acc[i][j] = fmaf(a[i].w, b[j].w, acc[i][j]);
            }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int r = ty + 16 * i, c = tx + 8 * j;
            const long long q = q0 + r, k = k0 + c;
            bool ok = k <= q;                                   // causal (also covers k < L since q < L)
            if (visit == 1) ok = ok && (q - k <= w0);           // local window, R1: q-k <= w0
            if (visit == 2) ok = ok && (q - k > w0);
            sm.s[r * (BN + 1) + c] = ok ? acc[i][j] * scale : -INFINITY;
        }
}

// online softmax on sm.s: 2 threads per row; writes p back into sm.s, alpha/m/l into smem
template <int D> __device__ inline void softmax_tile(Smem<D>& sm, int tid) {
    const int r = tid >> 1, hf = tid & 1;
    float* srow = &sm.s[r * (BN + 1) + hf * 32];
    float mx = -INFINITY;
#pragma unroll 8
    for (int c = 0; c < 32; ++c) mx = fmaxf(mx, srow[c]);
    mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
    const float m_old = sm.m[r];
    const float m_new = fmaxf(m_old, mx);
    float sum = 0.f;
    if (m_new == -INFINITY) {                                    // row fully masked so far
#pragma unroll 8
        for (int c = 0; c < 32; ++c) srow[c] = 0.f;
    } else {
#pragma unroll 8
        for (int c = 0; c < 32; ++c) {
            const float p = expf(srow[c] - m_new);               // exp(-inf) = 0 for masked entries
            srow[c] = p;
            sum += p;
        }
    }
    sum += __shfl_xor_sync(0xffffffffu, sum, 1);
    __syncwarp();
    if (hf == 0) {
        const float a = (m_new == -INFINITY) ? 1.f : expf(m_old - m_new);   // m_old = -inf -> 0
        sm.alpha[r] = a;
        sm.l[r] = sm.l[r] * a + sum;
        sm.m[r] = m_new;
    }
}

template <typename T, int D, bool BIFOCAL>
__global__ void __launch_bounds__(NT) prefill_simt_kernel(const T* __restrict__ Q, const T* __restrict__ K,
                                                          const T* __restrict__ V, T* __restrict__ out,
                                                          float* __restrict__ lse, long long L, int H_q, int H_kv,
                                                          long long w0, const float2* __restrict__ tab) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem<D>& sm = *reinterpret_cast<Smem<D>*>(smem_raw);
    constexpr int LD = Smem<D>::LD, HALF = D / 2;
    const int tid = threadIdx.x;
    const long long n_qt = (L + BM - 1) / BM;
    const long long qt = n_qt - 1 - blockIdx.x;                  // heaviest tiles first
    const int h = blockIdx.y, kv = h / (H_q / H_kv);
    const long long q0 = qt * BM;
    const float scale = 1.0f / sqrtf((float)D);

    // ---- load Q tile, build Q' = R(Delta q) Q (step a4) -------------------------------------------------
    for (int idx = tid; idx < BM * D; idx += NT) {
        const int r = idx / D, c = idx - r * D;
        const long long q = q0 + r;
        sm.q[r * LD + c] = q < L ? to_f32<T>(Q[((size_t)q * H_q + h) * D + c]) : 0.f;
    }
    if (tid < BM) { sm.m[tid] = -INFINITY; sm.l[tid] = 0.f; sm.alpha[tid] = 1.f; }
    __syncthreads();
    if (BIFOCAL) {
        for (int idx = tid; idx < BM * HALF; idx += NT) {
            const int r = idx / HALF, i = idx - r * HALF;
            const long long q = q0 + r;
            float2 cs = q < L ? tab[(size_t)q * HALF + i] : make_float2(1.f, 0.f);
            const float x1 = sm.q[r * LD + i], x2 = sm.q[r * LD + i + HALF];
            sm.qr[r * LD + i] = x1 * cs.x - x2 * cs.y;
            sm.qr[r * LD + i + HALF] = x1 * cs.y + x2 * cs.x;
        }
    }
    const int ty = tid >> 3, tx = tid & 7;
    constexpr int CPT = D / 8;                                   // O columns per thread: tx*CPT ..
    float o[4][CPT];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int c = 0; c < CPT; ++c) o[i][c] = 0.f;

    const long long q_last = (q0 + BM - 1 < L - 1) ? q0 + BM - 1 : L - 1;
    const long long n_kt = q_last / BN + 1;
    for (long long kt = 0; kt < n_kt; ++kt) {
        const long long k0 = kt * BN;
        __syncthreads();                                         // previous tile fully consumed
        for (int idx = tid; idx < BN * D; idx += NT) {
            const int r = idx / D, c = idx - r * D;
            const long long k = k0 + r;
            const size_t g = ((size_t)k * H_kv + kv) * D + c;
            sm.k[r * LD + c] = k < L ? to_f32<T>(K[g]) : 0.f;
            sm.v[r * D + c] = k < L ? to_f32<T>(V[g]) : 0.f;
        }
        __syncthreads();
        // step a3: classify.  local elements exist iff min(q-k) <= w0; remote iff max(q-k) > w0
        bool has_local = true, has_remote = false;
        if (BIFOCAL) {
            has_local = (q0 - (k0 + BN - 1)) <= w0;
            has_remote = (q_last - k0) > w0;
        }
        for (int pass = 0; pass < 2; ++pass) {
            if (pass == 0 && !has_local) continue;
            if (pass == 1 && !has_remote) continue;
            if (pass == 1) {                                     // step a5: rotate the K tile in smem
                __syncthreads();
                for (int idx = tid; idx < BN * HALF; idx += NT) {
                    const int r = idx / HALF, i = idx - r * HALF;
                    const long long k = k0 + r;
                    if (k < L) {
                        const float2 cs = tab[(size_t)k * HALF + i];
                        const float x1 = sm.k[r * LD + i], x2 = sm.k[r * LD + i + HALF];
                        sm.k[r * LD + i] = x1 * cs.x - x2 * cs.y;
                        sm.k[r * LD + i + HALF] = x1 * cs.y + x2 * cs.x;
                    }
                }
                __syncthreads();
            }
            const int visit = !BIFOCAL ? 0 : (pass == 0 ? 1 : 2);
            qk_tile<D>(sm, pass == 0 ? sm.q : sm.qr, tid, scale, q0, k0, w0, visit);     // step a6
            __syncthreads();
            softmax_tile<D>(sm, tid);
            __syncthreads();
            float al[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) al[i] = sm.alpha[ty + 16 * i];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int c = 0; c < CPT; ++c) o[i][c] *= al[i];
#pragma unroll 4
            for (int j = 0; j < BN; ++j) {
                float p[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) p[i] = sm.s[(ty + 16 * i) * (BN + 1) + j];
#pragma unroll
                for (int c = 0; c < CPT; c += 4) {
                    const float4 vv = *reinterpret_cast<const float4*>(&sm.v[j * D + tx * CPT + c]);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        o[i][c] = fmaf(p[i], vv.x, o[i][c]);
                        o[i][c + 1] = fmaf(p[i], vv.y, o[i][c + 1]);
                        o[i][c + 2] = fmaf(p[i], vv.z, o[i][c + 2]);
                        o[i][c + 3] = fmaf(p[i], vv.w, o[i][c + 3]);
                    }
                }
            }
        }
    }
    __syncthreads();
    // ---- epilogue (step a8): out = O / l, lse = m + ln l ------------------------------------------------
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = ty + 16 * i;
        const long long q = q0 + r;
        if (q >= L) continue;
        const float inv = 1.f / sm.l[r];
#pragma unroll
        for (int c = 0; c < CPT; ++c) out[((size_t)q * H_q + h) * D + tx * CPT + c] = from_f32<T>(o[i][c] * inv);
        if (tx == 0) lse[(size_t)h * L + q] = sm.m[r] + logf(sm.l[r]);
    }
}

template <typename T, int D, bool B>
int launch_t(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q, int H_kv,
             long long w0, const float2* tab, cudaStream_t st) {
    auto kern = prefill_simt_kernel<T, D, B>;
    const size_t smem = sizeof(Smem<D>);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return check_launch("prefill_simt attr");
    dim3 grid((unsigned)((L + BM - 1) / BM), (unsigned)H_q);
    kern<<<grid, NT, smem, st>>>((const T*)Q, (const T*)K, (const T*)V, (T*)out, lse, L, H_q, H_kv, w0, tab);
    note_launch();
    return check_launch("prefill_simt_kernel");
}

}  // namespace

int launch_prefill_simt(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                        int H_kv, int d, long long w0, long long G, const float2* tab, int dtype, bool bifocal,
                        cudaStream_t st) {
    (void)G;
#define JL_GO(T, D)                                                                                    \
    return bifocal ? launch_t<T, D, true>(Q, K, V, out, lse, L, H_q, H_kv, w0, tab, st)              \
                   : launch_t<T, D, false>(Q, K, V, out, lse, L, H_q, H_kv, w0, tab, st)
    if (dtype == JETLONG_FP32) {
        if (d == 64) { JL_GO(float, 64); }
        JL_GO(float, 128);
    }
    if (d == 64) { JL_GO(__nv_bfloat16, 64); }
    JL_GO(__nv_bfloat16, 128);
#undef JL_GO
}

}  // namespace jetlong
