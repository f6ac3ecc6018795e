// prefill_v2.cuh -- host interface of the two-tile tcgen05 prefill kernel (prefill_umma2.cu).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace jetlong {

struct PrefillV2Args {
    CUtensorMap tmQ;                                  // Q (or Q' fp16) [L, H_q, 128], box 64 channels x 1 head x 128 rows
    CUtensorMap tmK, tmV;                             // stored K (box 64 x 1 x 64 rows), V (box 64 x 1 x 128 rows)
    CUtensorMap tmKh, tmKe, tmKl;                     // workspace variant: K'hi fp16, K' e5m2 / compact rows, K'lo e5m2
    void* out;                                        // bf16 [L, H_q, 128], or fp32 when out_f32
    float* lse;
    long long L, w0, G;
    int H_q, H_kv;
    int bifocal;                                      // 0: control (every visit multiplies the stored operands)
    int precise;                                      // 0 fast, 2 full e5m2 cross terms, 3 selective e5m2 cross terms
    int prerot;                                       // remote K tiles come pre-rotated from the workspace (8(f)-1)
    int window_only;                                  // 1: only the local band on the stored operands (call A); 2: the band on the remote operands (call C)
    int out_f32;                                      // out holds fp32 (partial outputs of the unfused baseline)
    int qk_f16;                                       // Q and K hold fp16 (pre-rotated operands of calls B and C)
    const float2* lo;                                 // two-level (cos, sin) tables
    const float2* hi;
    const uint32_t* selinfo;                          // [H_kv][16] selective-compensation table (precise 3)
    int qb_lo = 0, qb_hi = -1;                        // query blocks [qb_lo, qb_hi) of this launch (multiples of 4; -1 = to the end):
                                                      // jetlong_prefill_host pipelines row chunks against the copies
};

// true when the two-tile kernel serves this precision mode (fp16 cross terms need the TMEM-resident Q of prefill_umma.cu)
inline bool prefill_v2_serves(int precise) { return precise == 0 || precise == 2 || precise == 3; }
int launch_prefill_v2(const PrefillV2Args& a, cudaStream_t st);

}  // namespace jetlong
