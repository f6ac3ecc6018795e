// api.cu -- the C ABI of libjetlong (include/jetlong.h): validation, dispatch, workspace layout.
#include <atomic>
#include <mutex>
#include <vector>
#include <stdio.h>
#include <string.h>

#include "common.cuh"

namespace jetlong {

static std::atomic<long long> g_launches{0};
static thread_local char g_err[256] = "no CUDA error recorded";
// per-thread defaults behind the deprecated setters; a call's jetlong_options override them
static thread_local int t_prefill_impl = -1;
static thread_local int t_prefill_precision = JETLONG_PRECISION_COMPENSATED;

static bool precision_known(int m) {
    return m == JETLONG_PRECISION_COMPENSATED || m == JETLONG_PRECISION_FAST || m == JETLONG_PRECISION_COMPENSATED_F16 ||
           m == JETLONG_PRECISION_COMPENSATED_E5M2;
}
struct Resolved { int precision, impl, map; double alpha, beta; bool ok; };
static Resolved resolve(const jetlong_options* opt) {
    Resolved r{t_prefill_precision, t_prefill_impl, JETLONG_MAP_ALIAS, 1.0, 32.0, true};
    if (opt) {
        if (opt->struct_bytes < sizeof(jetlong_options)) { r.ok = false; return r; }
        if (opt->precision != JETLONG_DEFAULT) r.precision = opt->precision;
        if (opt->prefill_impl != JETLONG_DEFAULT) r.impl = opt->prefill_impl;
        if (opt->remote_map != JETLONG_DEFAULT) r.map = opt->remote_map;
        if (opt->yarn_alpha != 0.0 || opt->yarn_beta != 0.0) { r.alpha = opt->yarn_alpha; r.beta = opt->yarn_beta; }
    }
    r.ok = precision_known(r.precision) && r.impl >= -1 && r.impl <= 4 &&
           (r.map == JETLONG_MAP_ALIAS || r.map == JETLONG_MAP_FREQ_INTERP) && r.beta > r.alpha;
    return r;
}
static FreqMap make_map(const Resolved& o, long long G, long long w_pre) {
    if (o.map != JETLONG_MAP_FREQ_INTERP) return alias_map();
    return FreqMap{1, 1.0 - 1.0 / (double)G, (double)w_pre, o.alpha, o.beta};
}

void note_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return JETLONG_OK;
    snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    return JETLONG_CUDA_ERROR;
}

// prefill_umma.cu
bool umma_prefill_supported(long long L, int H_q, int H_kv, int d, int dtype);
size_t umma_prefill_workspace_bytes(long long L, int H_q, int H_kv, int d);
size_t umma_prefill_prerot_workspace_bytes(long long L, int H_kv, int d);
size_t umma_prefill_unfused_workspace_bytes(long long L, int H_q, int H_kv, int d);
int launch_prefill_unfused(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                           int H_kv, int d, long long w0, long long G, double theta, void* ws, cudaStream_t st);
int launch_prefill_umma(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                        int H_kv, int d, long long w0, long long G, double theta, bool bifocal, int precise, void* ws,
                        size_t ws_bytes, cudaStream_t st, bool prerot, bool two_tile, FreqMap fm, int qb_lo, int qb_hi,
                        long long L_sel);

// decode.cu / decode_umma.cu
bool umma_decode_supported(int H_q, int H_kv, int d, int dtype);
bool umma_decode_paged_supported(int H_q, int H_kv, int d, int dtype);
size_t decode_paged_workspace_bytes(long long Lmax, int batch, int H_q, int H_kv, int d);
int launch_decode_paged(const void* q, const void* Kpool, const void* Vpool, const int* page_table, int max_pages,
                        long long pool_pages, const long long* Ls, const long long* Gs, int batch, void* out, float* lse,
                        int H_q, int H_kv, long long w0, double theta, void* ws, cudaStream_t st);

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static int validate(const void* a, const void* b, const void* c, const void* o, const void* l, long long L, int H_q,
                    int H_kv, int d, long long w0, long long w_pre, double theta, int dtype) {
    if (!a || !b || !c || !o || !l) return JETLONG_INVALID_ARG;
    if (L < 1 || H_q < 1 || H_kv < 1 || (H_q % H_kv) != 0) return JETLONG_INVALID_ARG;
    if (d != 64 && d != 128) return JETLONG_INVALID_ARG;
    if (w0 < 0 || w_pre < 1 || !(theta > 0.0)) return JETLONG_INVALID_ARG;
    if (dtype != JETLONG_BF16 && dtype != JETLONG_FP32) return JETLONG_INVALID_ARG;
    if (!aligned16(a) || !aligned16(b) || !aligned16(c) || !aligned16(o) || !aligned16(l)) return JETLONG_INVALID_ARG;
    return JETLONG_OK;
}

static int device_ok() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return JETLONG_UNSUPPORTED; }
    int major = 0, minor = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess) {
        cudaGetLastError();
        return JETLONG_UNSUPPORTED;
    }
    return (major == 10 && minor == 0) ? JETLONG_OK : JETLONG_UNSUPPORTED;   // the library carries sm_100a code only
}

static bool use_umma(int impl, long long L, int H_q, int H_kv, int d, int dtype) {
    if (impl == 0) return false;
    return umma_prefill_supported(L, H_q, H_kv, d, dtype);
}

static size_t prefill_ws(long long L, int H_q, int H_kv, int d, int dtype, bool bifocal) {
    size_t simt = bifocal ? align256((size_t)L * (d / 2) * sizeof(float2)) : 0;
    size_t umma = umma_prefill_supported(L, H_q, H_kv, d, dtype) ? umma_prefill_workspace_bytes(L, H_q, H_kv, d) : 0;
    return simt > umma ? simt : umma;      // either implementation may be selected at run time
}

static int prefill_common(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                          int H_kv, int d, long long w0, long long w_pre, double theta, int dtype, void* ws,
                          size_t ws_bytes, void* stream, bool bifocal, bool prerot = false,
                          const jetlong_options* opt = nullptr, int qb_lo = 0, int qb_hi = -1) {
    int rc = validate(Q, K, V, out, lse, L, H_q, H_kv, d, w0, w_pre, theta, dtype);
    if (rc != JETLONG_OK) return rc;
    const Resolved o = resolve(opt);
    if (!o.ok) return JETLONG_INVALID_ARG;
    if (prerot && !umma_prefill_supported(L, H_q, H_kv, d, dtype)) return JETLONG_UNSUPPORTED;
    long long G = bifocal ? jetlong_group_size(L, w_pre) : 1;
    if (G == 1 || w0 >= L - 1) bifocal = false;          // step a2: G = 1 (or an all-covering window) is the control
    const size_t need = (prerot && bifocal) ? umma_prefill_prerot_workspace_bytes(L, H_kv, d) : prefill_ws(L, H_q, H_kv, d, dtype, bifocal);
    if (need > 0 && (!ws || ws_bytes < need || !aligned16(ws))) return JETLONG_INVALID_ARG;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int prec = o.precision;
    const FreqMap fm = bifocal ? make_map(o, G, w_pre) : alias_map();
    if (fm.interp) G = kInterpG;                         // the kernels' form of the map: n = -Delta = x (common.cuh)
    if (prerot || use_umma(o.impl, L, H_q, H_kv, d, dtype))
        return launch_prefill_umma(Q, K, V, out, lse, L, H_q, H_kv, d, w0, G, theta, bifocal,
                                   prec == JETLONG_PRECISION_FAST ? 0 : prec == JETLONG_PRECISION_COMPENSATED_F16 ? 1 : prec == JETLONG_PRECISION_COMPENSATED_E5M2 ? 6 : 2,
                                   ws, ws_bytes, st,
                                   prerot && bifocal, /*two_tile=*/o.impl != 1 || qb_hi >= 0, fm, qb_lo, qb_hi,
                                   qb_hi >= 0 ? 128ll * qb_hi : L);
    const float2* tab = nullptr;
    if (bifocal) {
        rc = build_key_table((float2*)ws, L, G, d, theta, st, fm);
        if (rc != JETLONG_OK) return rc;
        tab = (const float2*)ws;
    }
    return launch_prefill_simt(Q, K, V, out, lse, L, H_q, H_kv, d, w0, G, tab, dtype, bifocal, st);
}

static int decode_common(const void* q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                         int H_kv, int d, long long w0, long long w_pre, double theta, int dtype, void* ws,
                         size_t ws_bytes, void* stream, bool bifocal, const jetlong_options* opt = nullptr) {
    int rc = validate(q, K, V, out, lse, L, H_q, H_kv, d, w0, w_pre, theta, dtype);
    if (rc != JETLONG_OK) return rc;
    const Resolved o = resolve(opt);
    if (!o.ok) return JETLONG_INVALID_ARG;
    long long G = bifocal ? jetlong_group_size(L, w_pre) : 1;
    if (G == 1 || w0 >= L - 1) bifocal = false;
    const FreqMap fm = bifocal ? make_map(o, G, w_pre) : alias_map();
    if (fm.interp) G = kInterpG;
    const size_t need = decode_workspace_bytes(L, H_q, H_kv, d);
    if (!ws || ws_bytes < need || !aligned16(ws)) return JETLONG_INVALID_ARG;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    return launch_decode(q, K, V, out, lse, L, H_q, H_kv, d, w0, G, theta, dtype, bifocal, ws, ws_bytes,
                         (cudaStream_t)stream, fm);
}

}  // namespace jetlong

using namespace jetlong;

extern "C" {

int64_t jetlong_group_size(int64_t L, int64_t w_pretrained) {
    if (L < 1 || w_pretrained < 1) return -1;
    int64_t G = (L + w_pretrained - 1) / w_pretrained;      // Eq.(2), integers only
    return G < 1 ? 1 : G;
}

size_t jetlong_workspace_bytes(int op, int64_t L, int H_q, int H_kv, int head_dim, int dtype) {
    if (L < 1 || H_q < 1 || H_kv < 1 || (H_q % H_kv) || (head_dim != 64 && head_dim != 128)) return 0;
    switch (op) {
        case JETLONG_OP_PREFILL: return prefill_ws(L, H_q, H_kv, head_dim, dtype, true);
        case JETLONG_OP_CAUSAL_PREFILL: return prefill_ws(L, H_q, H_kv, head_dim, dtype, false);
        case JETLONG_OP_DECODE:
        case JETLONG_OP_CAUSAL_DECODE: return decode_workspace_bytes(L, H_q, H_kv, head_dim);
        case JETLONG_OP_PREFILL_UNFUSED:
            return umma_prefill_supported(L, H_q, H_kv, head_dim, dtype) ? umma_prefill_unfused_workspace_bytes(L, H_q, H_kv, head_dim) : 0;
        case JETLONG_OP_PREFILL_PREROTATED:
            return umma_prefill_supported(L, H_q, H_kv, head_dim, dtype) ? umma_prefill_prerot_workspace_bytes(L, H_kv, head_dim) : 0;
        default: return 0;
    }
}

int jetlong_prefill(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q, int H_kv,
                    int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype, void* workspace,
                    size_t workspace_bytes, void* stream) {
    return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                          workspace, workspace_bytes, stream, true);
}

int jetlong_prefill_prerotated(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q,
                               int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                               void* workspace, size_t workspace_bytes, void* stream) {
    return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                          workspace, workspace_bytes, stream, true, true);
}

int jetlong_prefill_opt(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q, int H_kv,
                        int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype, void* workspace,
                        size_t workspace_bytes, void* stream, const jetlong_options* options) {
    return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                          workspace, workspace_bytes, stream, true, false, options);
}

int jetlong_prefill_prerotated_opt(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q,
                                   int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta,
                                   int dtype, void* workspace, size_t workspace_bytes, void* stream,
                                   const jetlong_options* options) {
    return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                          workspace, workspace_bytes, stream, true, true, options);
}

int jetlong_prefill_unfused(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q,
                            int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                            void* workspace, size_t workspace_bytes, void* stream) {
    int rc = validate(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype);
    if (rc != JETLONG_OK) return rc;
    if (!umma_prefill_supported(L, H_q, H_kv, head_dim, dtype)) return JETLONG_UNSUPPORTED;
    const long long G = jetlong_group_size(L, w_pretrained);
    if (G == 1 || w_local >= L - 1)                          // nothing is remote: the control, as in jetlong_prefill
        return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                              workspace, workspace_bytes, stream, true);
    const size_t need = umma_prefill_unfused_workspace_bytes(L, H_q, H_kv, head_dim);
    if (!workspace || workspace_bytes < need || !aligned16(workspace)) return JETLONG_INVALID_ARG;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    return launch_prefill_unfused(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, G, rope_theta, workspace,
                                  (cudaStream_t)stream);
}

int jetlong_causal_prefill(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q,
                           int H_kv, int head_dim, int dtype, void* workspace, size_t workspace_bytes, void* stream) {
    return prefill_common(Q, K, V, out, lse, L, H_q, H_kv, head_dim, 0, 1, 1.0, dtype, workspace, workspace_bytes,
                          stream, false);
}

int jetlong_decode(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse, int64_t L, int H_q,
                   int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                   void* workspace, size_t workspace_bytes, void* stream) {
    return decode_common(q, Kcache, Vcache, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                         workspace, workspace_bytes, stream, true);
}

int jetlong_decode_opt(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse, int64_t L, int H_q,
                       int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                       void* workspace, size_t workspace_bytes, void* stream, const jetlong_options* options) {
    return decode_common(q, Kcache, Vcache, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype,
                         workspace, workspace_bytes, stream, true, options);
}

size_t jetlong_decode_paged_workspace_bytes(int64_t max_len, int batch, int H_q, int H_kv, int head_dim) {
    if (max_len < 1 || batch < 1 || H_q < 1 || H_kv < 1 || (H_q % H_kv) || head_dim != 128) return 0;
    return decode_paged_workspace_bytes(max_len, batch, H_q, H_kv, head_dim);
}

int jetlong_decode_paged(const void* q, const void* Kpool, const void* Vpool, const int32_t* page_table,
                         const int64_t* seq_lens, int batch, int max_pages_per_seq, int64_t pool_pages, void* out, float* lse,
                         int H_q, int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                         void* workspace, size_t workspace_bytes, void* stream) {
    if (!page_table || !seq_lens || batch < 1 || max_pages_per_seq < 1 || pool_pages < 1) return JETLONG_INVALID_ARG;
    int rc = validate(q, Kpool, Vpool, out, lse, 1, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype);
    if (rc != JETLONG_OK) return rc;
    long long Lmax = 0;
    std::vector<long long> Ls(batch), Gs(batch);
    for (int b = 0; b < batch; ++b) {
        if (seq_lens[b] < 1 || seq_lens[b] > 128ll * max_pages_per_seq) return JETLONG_INVALID_ARG;
        Ls[b] = seq_lens[b];
        Gs[b] = jetlong_group_size(seq_lens[b], w_pretrained);       // Eq.(2) per sequence, on the host
        if (Ls[b] > Lmax) Lmax = Ls[b];
    }
    if (!umma_decode_paged_supported(H_q, H_kv, head_dim, dtype)) return JETLONG_UNSUPPORTED;
    const size_t need = decode_paged_workspace_bytes(Lmax, batch, H_q, H_kv, head_dim);
    if (!workspace || workspace_bytes < need || !aligned16(workspace)) return JETLONG_INVALID_ARG;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    return launch_decode_paged(q, Kpool, Vpool, page_table, max_pages_per_seq, pool_pages, Ls.data(), Gs.data(), batch, out,
                               lse, H_q, H_kv, w_local, rope_theta, workspace, (cudaStream_t)stream);
}

// ---- allocation-free decode (include/jetlong.h) --------------------------------------------------------------------
// The scratch of jetlong_decode_static.  In host code this name is only a handle for the runtime, NOT a device address:
// the address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[JETLONG_STATIC_SCRATCH_BYTES];
static void* g_static_ptr[64];
static std::mutex g_static_mu;

static int static_scratch(void** ws) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess && (dev < 0 || dev >= 64)) e = cudaErrorInvalidDevice;
    if (e == cudaSuccess) {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_ptr[dev]) {
            void* ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_static_scratch);
            if (e == cudaSuccess && !ptr) e = cudaErrorInvalidSymbol;
            if (e == cudaSuccess) g_static_ptr[dev] = ptr;
        }
        *ws = g_static_ptr[dev];
    }
    if (e != cudaSuccess) {
        snprintf(g_err, sizeof(g_err), "jetlong_decode_static: address of the static scratch: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return JETLONG_CUDA_ERROR;
    }
    return JETLONG_OK;
}

int jetlong_decode_static_init(void) {
    int rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    void* ws = nullptr;
    return static_scratch(&ws);
}

int jetlong_decode_static(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse, int64_t L, int H_q,
                          int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype,
                          void* stream) {
    int rc = validate(q, Kcache, Vcache, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype);
    if (rc != JETLONG_OK) return rc;
    if (decode_workspace_bytes(L, H_q, H_kv, head_dim) > (size_t)JETLONG_STATIC_SCRATCH_BYTES) return JETLONG_SCRATCH_EXCEEDED;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    void* ws = nullptr;
    rc = static_scratch(&ws);
    if (rc != JETLONG_OK) return rc;
    return decode_common(q, Kcache, Vcache, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype, ws,
                         (size_t)JETLONG_STATIC_SCRATCH_BYTES, stream, true);
}

int jetlong_causal_decode(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse, int64_t L,
                          int H_q, int H_kv, int head_dim, int dtype, void* workspace, size_t workspace_bytes,
                          void* stream) {
    return decode_common(q, Kcache, Vcache, out, lse, L, H_q, H_kv, head_dim, 0, 1, 1.0, dtype, workspace,
                         workspace_bytes, stream, false);
}

// staging arena of jetlong_prefill_host: one per device, grown on demand, reused from call to call
struct HostArena {
    unsigned char* base = nullptr;
    size_t bytes = 0;
    cudaStream_t st = nullptr, st_in = nullptr, st_out = nullptr;   // compute, host-to-device, device-to-host
    cudaEvent_t ev_in[16] = {}, ev_done[16] = {};
};
static HostArena g_arena[64];
static std::mutex g_arena_mu;

void jetlong_host_release(void) {
    std::lock_guard<std::mutex> lock(g_arena_mu);
    int cur = 0;
    cudaGetDevice(&cur);
    for (int d = 0; d < 64; ++d) {
        HostArena& a = g_arena[d];
        if (!a.base && !a.st) continue;
        cudaSetDevice(d);
        if (a.base) cudaFree(a.base);
        if (a.st) cudaStreamDestroy(a.st);
        if (a.st_in) cudaStreamDestroy(a.st_in);
        if (a.st_out) cudaStreamDestroy(a.st_out);
        for (int i = 0; i < 16; ++i) { if (a.ev_in[i]) cudaEventDestroy(a.ev_in[i]); if (a.ev_done[i]) cudaEventDestroy(a.ev_done[i]); }
        a = HostArena();
    }
    cudaSetDevice(cur);
    cudaGetLastError();
}

int jetlong_prefill_host(const void* Q, const void* K, const void* V, void* out, float* lse, int64_t L, int H_q,
                         int H_kv, int head_dim, int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype) {
    int rc = validate(Q, K, V, out, lse, L, H_q, H_kv, head_dim, w_local, w_pretrained, rope_theta, dtype);
    if (rc != JETLONG_OK) return rc;
    rc = device_ok();
    if (rc != JETLONG_OK) return rc;
    const size_t es = dtype == JETLONG_FP32 ? 4 : 2;
    const size_t rq = (size_t)H_q * head_dim * es, rk = (size_t)H_kv * head_dim * es;   // bytes per row
    const size_t nq = (size_t)L * rq, nk = (size_t)L * rk;
    const size_t nl = (size_t)L * H_q * sizeof(float);
    const size_t nws = jetlong_workspace_bytes(JETLONG_OP_PREFILL, L, H_q, H_kv, head_dim, dtype);
    const size_t oq = 0, ok = align256(nq), ov = ok + align256(nk), oo = ov + align256(nk), ol = oo + align256(nq),
                 ow = ol + align256(nl), total = ow + align256(nws) + 256;
    int devid = 0;
    if (cudaGetDevice(&devid) != cudaSuccess || devid < 0 || devid >= 64) return check_launch("cudaGetDevice");
    std::lock_guard<std::mutex> lock(g_arena_mu);               // calls are serialised: they share the arena
    HostArena& a = g_arena[devid];
    if (!a.st) {
        if (cudaStreamCreateWithFlags(&a.st, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&a.st_in, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&a.st_out, cudaStreamNonBlocking) != cudaSuccess)
            return check_launch("cudaStreamCreate");
        for (int i = 0; i < 16; ++i)
            if (cudaEventCreateWithFlags(&a.ev_in[i], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&a.ev_done[i], cudaEventDisableTiming) != cudaSuccess)
                return check_launch("cudaEventCreate");
    }
    if (a.bytes < total) {
        if (a.base && cudaFree(a.base) != cudaSuccess) return check_launch("cudaFree");
        a.base = nullptr; a.bytes = 0;
        if (cudaMalloc(&a.base, total) != cudaSuccess) return check_launch("cudaMalloc");
        a.bytes = total;
    }
    unsigned char* dev = a.base;
    // the table header must start zeroed (jetlong_workspace_bytes contract); the region moves with the shapes, so every call
    if (cudaMemsetAsync(dev + ow, 0, 256, a.st) != cudaSuccess) return check_launch("cudaMemsetAsync");
    // Row chunks, ascending: rows [r0, r1) need only keys < r1, so chunk c can run as soon as ITS rows of K, V, Q are on the
    // device; its out / lse rows go back while the next chunk runs.  The tcgen05 two-tile kernel launches by row range
    // (multiples of 512 rows); other shapes run as one chunk.
    int nch = 1;
    if (umma_prefill_supported(L, H_q, H_kv, head_dim, dtype) && L >= 8192) nch = L >= 32768 ? 8 : 4;
    long long step = ((L + nch - 1) / nch + 511) / 512 * 512;
    bool ok_all = true;
    for (int c = 0; c < nch && ok_all; ++c) {
        const long long r0 = c * step, r1 = (c + 1 == nch || (c + 1) * step > L) ? L : (c + 1) * step;
        if (r0 >= L) { nch = c; break; }
        const size_t n = (size_t)(r1 - r0);
        ok_all = cudaMemcpyAsync(dev + ok + r0 * rk, (const unsigned char*)K + r0 * rk, n * rk, cudaMemcpyHostToDevice, a.st_in) == cudaSuccess &&
                 cudaMemcpyAsync(dev + ov + r0 * rk, (const unsigned char*)V + r0 * rk, n * rk, cudaMemcpyHostToDevice, a.st_in) == cudaSuccess &&
                 cudaMemcpyAsync(dev + oq + r0 * rq, (const unsigned char*)Q + r0 * rq, n * rq, cudaMemcpyHostToDevice, a.st_in) == cudaSuccess &&
                 cudaEventRecord(a.ev_in[c], a.st_in) == cudaSuccess;
        if (r1 == L) { nch = c + 1; break; }
    }
    if (!ok_all) { cudaStreamSynchronize(a.st_in); return check_launch("jetlong_prefill_host H2D"); }
    for (int c = 0; c < nch; ++c) {
        const long long r0 = c * step, r1 = (c + 1 == nch) ? L : (c + 1) * step;
        if (cudaStreamWaitEvent(a.st, a.ev_in[c], 0) != cudaSuccess) { rc = check_launch("cudaStreamWaitEvent"); break; }
        rc = prefill_common(dev + oq, dev + ok, dev + ov, dev + oo, (float*)(dev + ol), L, H_q, H_kv, head_dim, w_local,
                            w_pretrained, rope_theta, dtype, dev + ow, align256(nws) + 256, a.st, true, false, nullptr,
                            nch > 1 ? (int)(r0 / 128) : 0, nch > 1 ? (int)((r1 + 127) / 128) : -1);
        if (rc != JETLONG_OK) break;
        const size_t n = (size_t)(r1 - r0);
        if (cudaEventRecord(a.ev_done[c], a.st) != cudaSuccess || cudaStreamWaitEvent(a.st_out, a.ev_done[c], 0) != cudaSuccess ||
            cudaMemcpyAsync((unsigned char*)out + r0 * rq, dev + oo + r0 * rq, n * rq, cudaMemcpyDeviceToHost, a.st_out) != cudaSuccess ||
            cudaMemcpy2DAsync(lse + r0, (size_t)L * 4, (float*)(dev + ol) + r0, (size_t)L * 4, n * 4, (size_t)H_q,
                              cudaMemcpyDeviceToHost, a.st_out) != cudaSuccess) {
            rc = check_launch("jetlong_prefill_host D2H");
            break;
        }
    }
    const bool s1 = cudaStreamSynchronize(a.st) == cudaSuccess, s2 = cudaStreamSynchronize(a.st_out) == cudaSuccess,
               s3 = cudaStreamSynchronize(a.st_in) == cudaSuccess;
    if (rc == JETLONG_OK && !(s1 && s2 && s3)) rc = check_launch("jetlong_prefill_host");
    return rc;
}

const char* jetlong_status_string(int status) {
    switch (status) {
        case JETLONG_OK: return "ok";
        case JETLONG_INVALID_ARG: return "invalid argument";
        case JETLONG_UNSUPPORTED: return "unsupported device or configuration (needs compute capability 10.0, sm_100a)";
        case JETLONG_CUDA_ERROR: return g_err;
        case JETLONG_SCRATCH_EXCEEDED:
            return "the call needs more scratch than the library's static array holds (JETLONG_STATIC_SCRATCH_BYTES = 8 MiB): "
                   "use jetlong_decode with a caller-provided workspace";
        default: return "unknown status";
    }
}

int64_t jetlong_launch_count(void) { return g_launches.load(); }

int jetlong_set_prefill_impl(int impl) {
    const int prev = t_prefill_impl;
    if (impl >= -1 && impl <= 4) t_prefill_impl = (impl == 2 || impl == 3) ? 1 : impl;   // 2, 3: the removed cluster launches
    return prev;
}

int jetlong_set_prefill_precision(int mode) {
    const int prev = t_prefill_precision;
    if (precision_known(mode)) t_prefill_precision = mode;
    return prev;
}

int jetlong_prefill_uses_umma(int64_t L, int H_q, int H_kv, int head_dim) {
    return use_umma(t_prefill_impl, L, H_q, H_kv, head_dim, JETLONG_BF16) ? 1 : 0;
}

}  // extern "C"
