/*
 * jetlong.h -- C ABI of libjetlong: fused bifocal RoPE attention (Jet-Long,
 * arxiv/paper_2607_07740) for NVIDIA B200 (sm_100a).
 *
 * "P:nnn" cites a line of the paper text.  R1..R16 are the readings listed in
 * DESIGN.md for points the paper leaves open.
 *
 * Conventions common to every entry point
 *   - All tensor pointers are DEVICE pointers owned by the caller.  The library never allocates,
 *     frees or retains them.  Calls are asynchronous on `stream` (a cudaStream_t passed as void*).
 *   - Layouts (contiguous): Q, out [L, H_q, d]; K, V [L, H_kv, d]; lse [H_q, L] fp32.
 *     Decode: q, out [H_q, d]; lse [H_q]; Kcache, Vcache [>=L, H_kv, d] (rows 0..L-1 are read).
 *   - Q and K arrive ALREADY RoPE-rotated at their true absolute positions 0..L-1, half-split
 *     pairing (i, i+d/2), theta_i = rope_theta^(-2i/d)  (Eq.(4); q_local in Eq.(6); R5, R6).
 *     The library never writes to Q, K, V (the cache invariant).
 *   - softmax scale is 1/sqrt(head_dim) (R7); lse is the natural log of sum exp(scaled score) (R8).
 *   - GQA: query head h reads KV head h / (H_q / H_kv) (R9).
 *   - dtype: JETLONG_BF16 (bf16 Q/K/V/out, fp32 accumulation) or JETLONG_FP32 (fp32 everything).
 *   - Return value: a jetlong_status.  Arguments are validated before any launch; on a non-OK
 *     status nothing has been written.  There is no CPU fallback: without a compute-capability
 *     10.0 device (B200, sm_100a) the compute entry points return JETLONG_UNSUPPORTED.
 *   - Value range (bf16 path): rotated remote operands are re-rounded to fp16 and e5m2 for the tensor core, so
 *     |Q|, |K| elements must stay below 2^15 (a rotated pair can grow by sqrt 2; fp16 overflows at 65504, e5m2 at
 *     61440).  Larger magnitudes give inf / NaN remote scores; activations of the models in scope are < 2^10.
 *     Precision of the default mode: a frequency pair that is loud in Q AND in K at once (product of the
 *     two factors, relative to the other channels' rms, above ~12) is detected per KV head and its cross terms are kept
 *     in fp16; the lse error then reaches the tolerance (measured up to 9.8e-4 against 1e-3).  For such data
 *     JETLONG_PRECISION_COMPENSATED_F16 (4e-5, slower) can be chosen per call.
 *   - INVALID_ARG: null pointer, L < 1, H_q % H_kv != 0, head_dim not in {64, 128}, w_local < 0,
 *     w_pretrained < 1, rope_theta <= 0, unknown dtype, a pointer not 16-byte aligned, or a
 *     workspace smaller than jetlong_workspace_bytes() reports.
 */
#ifndef JETLONG_H_
#define JETLONG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    JETLONG_OK = 0,
    JETLONG_INVALID_ARG = 1,
    JETLONG_UNSUPPORTED = 2,
    JETLONG_CUDA_ERROR = 3,
    JETLONG_SCRATCH_EXCEEDED = 4     /* jetlong_decode_static only: the call needs more than JETLONG_STATIC_SCRATCH_BYTES */
} jetlong_status;

enum { JETLONG_BF16 = 0, JETLONG_FP32 = 1 };

/* op codes for jetlong_workspace_bytes */
enum { JETLONG_OP_PREFILL = 0, JETLONG_OP_DECODE = 1, JETLONG_OP_CAUSAL_PREFILL = 2, JETLONG_OP_CAUSAL_DECODE = 3,
       JETLONG_OP_PREFILL_PREROTATED = 4, JETLONG_OP_PREFILL_UNFUSED = 5 };

/* Eq.(2): G = max(1, ceil(L / w_pretrained)), integer arithmetic on the host.
 * Returns -1 if L < 1 or w_pretrained < 1. */
int64_t jetlong_group_size(int64_t L, int64_t w_pretrained);

/* Bytes of caller-allocated device workspace the op needs for these shapes (0 is possible).
 * Holds rotation tables (Eq.(5)-(6)) and split-KV partial states (decode).  16-byte aligned.
 * Contract: the first 256 bytes are a table header.  A workspace must be ZERO-FILLED before its first use (at least
 * its first 256 bytes); between calls that reuse it the caller must not write into it.  A sealed header
 * (magic, rope_theta, table length, head_dim, checksum of the table's first and last rows) lets consecutive calls
 * skip the table rebuild; a header that does not verify is rebuilt, never trusted. */
size_t jetlong_workspace_bytes(int op, int64_t L, int H_q, int H_kv, int head_dim, int dtype);

/*
 * Bifocal prefill (Eq.(1) P:70 with Eq.(2),(3),(5),(6); Section 3.3).
 * For every head h and row q: keys with 0 <= q-k <= w_local score with the stored Q, K (R1);
 * older keys score with R(Delta q) Q[q] and R(Delta k) K[k], Delta(x) = floor(x/G) - x, one G
 * from the full L (R3).  One joint softmax over k <= q.  The remote-only partial state replaces
 * the paper's (B - C), so no subtraction occurs (the merge is the additive LSE merge of Eq.(7)).
 * G == 1 dispatches to jetlong_causal_prefill: bitwise the control's result.
 */
int jetlong_prefill(const void* Q, const void* K, const void* V, void* out, float* lse,
                    int64_t L, int H_q, int H_kv, int head_dim,
                    int64_t w_local, int64_t w_pretrained, double rope_theta,
                    int dtype, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Workspace variant of the bifocal prefill (an ablation that prices the on-the-fly key correction; the paper
 * keeps "no second key view").  Same arguments and result as jetlong_prefill, but the correction
 * rotation K' = R(Delta k) K (Eq.(5)-(6) P:101-106) is applied ONCE into a scratch inside the workspace
 * (K' as fp16 plus the two e5m2 cross-term operands: 4 bytes per key channel, e.g. 268 MB at L = 65536,
 * H_kv = 8) and the remote tiles are then TMA-loaded from it; the stored K is still never written.
 * bf16, head_dim 128 only (JETLONG_UNSUPPORTED otherwise; any GQA group size); the workspace must be at
 * least jetlong_workspace_bytes(JETLONG_OP_PREFILL_PREROTATED, ...).  The fp16 cross-term precision
 * mode is served with the e5m2 cross terms.
 */
int jetlong_prefill_prerotated(const void* Q, const void* K, const void* V, void* out, float* lse,
                               int64_t L, int H_q, int H_kv, int head_dim,
                               int64_t w_local, int64_t w_pretrained, double rope_theta,
                               int dtype, void* workspace, size_t workspace_bytes, void* stream);

/*
 * The paper's UNFUSED procedure on the GPU (Section 3.3, "Jet-Long (unfused)" of Table 7), a baseline
 * for the fused kernel, never the product path: three launches of the same tcgen05 attention kernel --
 *   A: sliding-window attention (0 <= q-k <= w_local) on the stored Q, K;
 *   B: full causal attention at the remote positions, Q' = R(Delta q) Q, K' = R(Delta k) K;
 *   C: sliding-window attention at the remote positions --
 * each returning (O_X in fp32, l_X), then Eq.(7) WITH the minus sign in fp32:
 *   O = (W_A O_A + W_B O_B - W_C O_C) / (W_A + W_B - W_C).
 * K' is written once to the workspace (as in jetlong_prefill_prerotated); B and C score with the same compensated remote
 * operands as the fused kernel, so the baseline meets the same tolerances; the band is computed three times.
 * bf16, head_dim 128; workspace >= jetlong_workspace_bytes(JETLONG_OP_PREFILL_UNFUSED, ...)
 * (the workspace variant's region + O_A, O_B, O_C in fp32 + l_B, l_C: about 6.5x the size of Q).
 */
int jetlong_prefill_unfused(const void* Q, const void* K, const void* V, void* out, float* lse,
                            int64_t L, int H_q, int H_kv, int head_dim,
                            int64_t w_local, int64_t w_pretrained, double rope_theta,
                            int dtype, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Bifocal batch-1 decode: one query row per head at position L-1 against cache rows
 * 0..L-1 (the current token's key/value already appended at row L-1; R4, R14).  G is recomputed
 * from this L.  Split-KV scan; partial (m, l, O) states are merged by the additive LSE merge.
 */
int jetlong_decode(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse,
                   int64_t L, int H_q, int H_kv, int head_dim,
                   int64_t w_local, int64_t w_pretrained, double rope_theta,
                   int dtype, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Batched decode over a PAGED KV cache: `batch` independent sequences, one query token each
 * (Eq.(1) per sequence), in one launch per 16 sequences.  Sequence b has its own current length seq_lens[b]
 * (a HOST array; G_b = jetlong_group_size(seq_lens[b], w_pretrained) is computed on the host per sequence) and reads
 * its keys through a page table: logical rows [128 t, 128 t + 127] of sequence b live in physical page
 * page_table[b * max_pages_per_seq + t] of the pools Kpool, Vpool [pool_pages * 128, H_kv, d] (a page is the TMA tile
 * of the scan, so paging costs one table read per tile).  page_table is a DEVICE array of int32.  q, out [batch, H_q, d];
 * lse [batch, H_q].  Rows of a sequence's last page beyond its length are never used but must hold finite numbers.
 * bf16, head_dim 128, H_q / H_kv <= 16 (JETLONG_UNSUPPORTED otherwise); remote map: aliasing.
 * workspace >= jetlong_decode_paged_workspace_bytes(max over b of seq_lens[b], batch, ...), zero-filled before first use.
 * INVALID_ARG additionally: batch < 1, a length < 1 or > 128 * max_pages_per_seq, pool_pages < 1.
 */
size_t jetlong_decode_paged_workspace_bytes(int64_t max_len, int batch, int H_q, int H_kv, int head_dim);
int jetlong_decode_paged(const void* q, const void* Kpool, const void* Vpool, const int32_t* page_table,
                         const int64_t* seq_lens, int batch, int max_pages_per_seq, int64_t pool_pages,
                         void* out, float* lse, int H_q, int H_kv, int head_dim,
                         int64_t w_local, int64_t w_pretrained, double rope_theta,
                         int dtype, void* workspace, size_t workspace_bytes, void* stream);

/* Allocation-free decode.  The same operation and kernels as jetlong_decode (default options), for callers that cannot
 * allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  There is no
 * workspace argument: the rotation tables and the split partials live in ONE file-scope device array of
 * JETLONG_STATIC_SCRATCH_BYTES bytes inside the library (every GPU that loads the library holds these 8 MiB until the process
 * exits).  The entry point calls no cudaMalloc / cudaFree and no allocating library routine; the caller still passes q, the
 * cache, out and lse (device pointers, as for jetlong_decode).
 *   - Limit: jetlong_workspace_bytes(JETLONG_OP_DECODE, L, ...) <= JETLONG_STATIC_SCRATCH_BYTES, else
 *     JETLONG_SCRATCH_EXCEEDED and nothing is launched.  8 MiB cover L up to 1.5 M rows at H_q / H_kv = 32 / 8, d = 128
 *     (4.5 MB at L = 65536, 5.3 MB at 131072, 7.1 MB at 1 M: the partials of up to 2 x SMs splits, 520 B per
 *     (split, query head), and the tables at 512 B per 256 rows).
 *   - The array is shared by every call on the device and keeps the last call's contents.  Nothing in it has to start at
 *     zero per call: the table header is re-validated (parameters and a hash of the table body) and rebuilt when it does
 *     not fit the call, the partials are rewritten in full before they are read.
 *   - Calls that overlap on the GPU (two streams, two host threads on one device) RACE on the array: serialise them, or use
 *     jetlong_decode with one workspace per stream.
 * jetlong_decode_static_init() resolves the array's device address for the CURRENT device (cudaGetSymbolAddress, once per
 * device; JETLONG_CUDA_ERROR if that fails).  jetlong_decode_static does the same on its first call on a device; call the
 * init yourself before a stream capture starts, because the first use of the library on a device loads its module. */
#define JETLONG_STATIC_SCRATCH_BYTES (8u << 20)
int jetlong_decode_static_init(void);
int jetlong_decode_static(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse,
                          int64_t L, int H_q, int H_kv, int head_dim,
                          int64_t w_local, int64_t w_pretrained, double rope_theta,
                          int dtype, void* stream);

/* Matched control ("without bifocal attention"): plain causal attention on the given
 * (already RoPE'd) Q, K with the same kernels, no classifier and no rotation. */
int jetlong_causal_prefill(const void* Q, const void* K, const void* V, void* out, float* lse,
                           int64_t L, int H_q, int H_kv, int head_dim,
                           int dtype, void* workspace, size_t workspace_bytes, void* stream);

int jetlong_causal_decode(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse,
                          int64_t L, int H_q, int H_kv, int head_dim,
                          int dtype, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Host-buffer convenience wrappers (used for end-to-end timing): same arguments, but Q, K, V, out,
 * lse are HOST pointers (pinned or pageable).  The call copies in, runs the op, copies out / lse back and synchronises
 * before returning.  Device staging memory is taken from an arena the library keeps per device and reuses from call
 * to call (grown on demand, released by jetlong_host_release or at process exit); calls are serialised per device.
 * Every copy's status is checked (JETLONG_CUDA_ERROR).
 */
int jetlong_prefill_host(const void* Q, const void* K, const void* V, void* out, float* lse,
                         int64_t L, int H_q, int H_kv, int head_dim,
                         int64_t w_local, int64_t w_pretrained, double rope_theta, int dtype);

/* Frees the staging arenas of jetlong_prefill_host (all devices).  Safe to call at any time between calls. */
void jetlong_host_release(void);

/* Text for a status; for JETLONG_CUDA_ERROR the text of the last CUDA error seen by this thread. */
const char* jetlong_status_string(int status);

/* Number of kernels this process has launched through the library (for bench accounting). */
int64_t jetlong_launch_count(void);

/*
 * Per-call options of the prefill entry points (precision of the remote scores, implementation).  Pass NULL for the
 * defaults.  struct_bytes = sizeof(jetlong_options) (checked: a smaller value is JETLONG_INVALID_ARG); a field set to
 * JETLONG_DEFAULT takes the calling thread's default (see the two deprecated setters below).  Nothing in the library's
 * launch path is process-global: two host threads may call with different options on different streams.
 */
#define JETLONG_DEFAULT (-2)
typedef struct {
    uint32_t struct_bytes;
    int precision;      /* a JETLONG_PRECISION_* value or JETLONG_DEFAULT */
    int prefill_impl;   /* -1 / 4: tcgen05 two-tile kernel (default); 1: tcgen05 one-tile CTA pairs; 0: SIMT fp32; or JETLONG_DEFAULT */
    int remote_map;     /* JETLONG_MAP_ALIAS (0, the paper's method and the default) or JETLONG_MAP_FREQ_INTERP */
    double yarn_alpha;  /* ramp of JETLONG_MAP_FREQ_INTERP; 0, 0 = the YaRN defaults alpha = 1, beta = 32 */
    double yarn_beta;
} jetlong_options;

/* Remote map (Section 4.7, Table 6: "position aliasing (default Jet-Long) vs. YaRN-style frequency interpolation
 * within the same bifocal construction").  JETLONG_MAP_ALIAS is Eq.(3): remote position floor(x / G).
 * JETLONG_MAP_FREQ_INTERP is this library's DEFINITION of the ablation (the paper prints no formula; R17):
 * keys older than w_local score with RoPE at their TRUE positions but with the NTK-by-parts frequencies
 *     theta'_i = theta_i ((1 - gamma_i) / G + gamma_i),   gamma_i = clamp((w_pretrained theta_i / 2 pi - alpha) / (beta - alpha), 0, 1),
 * i.e. the stored operands are corrected by rotating pair i by -x (theta_i - theta'_i) at absolute position x; no extra
 * attention temperature (R10).  G = 1 is still the control.  Everything else (window rule, one joint softmax, cache
 * never written, precision modes) is unchanged.  Prefill (jetlong_prefill_opt, jetlong_prefill_prerotated_opt) and
 * decode (jetlong_decode_opt) accept it; the unfused baseline is aliasing only. */
enum { JETLONG_MAP_ALIAS = 0, JETLONG_MAP_FREQ_INTERP = 1 };

/* jetlong_prefill / jetlong_prefill_prerotated with explicit options; identical otherwise. */
int jetlong_prefill_opt(const void* Q, const void* K, const void* V, void* out, float* lse,
                        int64_t L, int H_q, int H_kv, int head_dim,
                        int64_t w_local, int64_t w_pretrained, double rope_theta,
                        int dtype, void* workspace, size_t workspace_bytes, void* stream,
                        const jetlong_options* options);
int jetlong_prefill_prerotated_opt(const void* Q, const void* K, const void* V, void* out, float* lse,
                                   int64_t L, int H_q, int H_kv, int head_dim,
                                   int64_t w_local, int64_t w_pretrained, double rope_theta,
                                   int dtype, void* workspace, size_t workspace_bytes, void* stream,
                                   const jetlong_options* options);

/* jetlong_decode with explicit options (only remote_map and the ramp are used). */
int jetlong_decode_opt(const void* q, const void* Kcache, const void* Vcache, void* out, float* lse,
                       int64_t L, int H_q, int H_kv, int head_dim,
                       int64_t w_local, int64_t w_pretrained, double rope_theta,
                       int dtype, void* workspace, size_t workspace_bytes, void* stream,
                       const jetlong_options* options);

/* DEPRECATED (kept as shims): set the CALLING THREAD's default prefill implementation.
 * -1 or 4 (default): tcgen05 UMMA where supported (bf16, head_dim 128, any GQA group size): the two-tile kernel, in which a
 * CTA pair owns 256 query rows x 2 heads and every staged / rotated K tile feeds both 128-row tiles (prefill_umma2.cu).
 * 1 = the one-tile CTA-pair kernel of round 1 (prefill_umma.cu, even group sizes; also serves JETLONG_PRECISION_COMPENSATED_F16);
 * 0 = SIMT fp32-FMA tiles.  2 and 3 (round 1's cluster-of-four launches, superseded by the two-tile kernel and
 * removed) are accepted and mean 1.  All give the same results up to rounding.  Returns the previous value. */
int jetlong_set_prefill_impl(int impl);

/* Operand precision of the REMOTE Q'K'^T on the tcgen05 prefill path.  Rotated operands must be
 * re-rounded for the tensor core; with one fp16 rounding (11 bits) the lse error reaches ~3e-3 on outlier-channel
 * inputs (tolerance 1e-3).  With y = hi + lo (hi = fp16(y), lo = y - hi):
 *   COMPENSATED (default): S = Q'hi K'hi (fp16 UMMA) + Q' K'lo + Q'lo K' with the two cross terms in e5m2
 *                          (kind::f8f6f4) over the two highest-energy channel pairs of every 8-pair chunk (32 of the
 *                          128 channels, chosen per KV head on the device from the pair energies of K and Q); a head
 *                          whose remaining channels are too loud (predicted score noise > 3e-4) gets the full cross
 *                          terms.  lse error 1e-4 (64K-128K) to 8e-4 (short, peaked rows).
 *   COMPENSATED_E5M2:      the two e5m2 cross terms over all 128 channels for every head; lse error ~3e-4.
 *   COMPENSATED_F16:       the two cross terms in fp16 (three fp16 UMMA groups, one-tile kernel); lse error ~1e-5.  The
 *                          workspace variant serves this mode with COMPENSATED_E5M2.
 *   FAST:                  Q'hi K'hi only; lse error up to ~3e-3 on such inputs (out still within tolerance).
 * Local tiles, the control and decode are unaffected (decode always compensates: fp16 K'hi [Q'hi; Q'lo] + e5m2 K'lo Q'hi).
 * DEPRECATED setter (a shim): sets the CALLING THREAD's default; prefer jetlong_options.precision.
 * Returns the previous mode; an unknown mode changes nothing. */
enum { JETLONG_PRECISION_COMPENSATED = 0, JETLONG_PRECISION_FAST = 1, JETLONG_PRECISION_COMPENSATED_F16 = 2,
       JETLONG_PRECISION_COMPENSATED_E5M2 = 3 };
int jetlong_set_prefill_precision(int mode);

/* 1 if a bf16 prefill of these shapes runs on the tcgen05 UMMA kernel under the current setting, else 0. */
int jetlong_prefill_uses_umma(int64_t L, int H_q, int H_kv, int head_dim);

#ifdef __cplusplus
}
#endif
#endif /* JETLONG_H_ */
