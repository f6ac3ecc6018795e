// common.cuh -- small shared device/host helpers of libjetlong (sm_100a only).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/jetlong.h"

namespace jetlong {

// launch accounting (jetlong_launch_count) and last CUDA error text (jetlong_status_string)
void note_launch(int n = 1);
int check_launch(const char* what);   // returns JETLONG_OK or JETLONG_CUDA_ERROR

// Delta(x) = floor(x/G) - x, Eq.(5) P:101 (x >= 0)
__host__ __device__ inline long long delta_pos(long long x, long long G) { return x / G - x; }

template <typename T> __device__ inline float to_f32(T v);
template <> __device__ inline float to_f32<float>(float v) { return v; }
template <> __device__ inline float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }

template <typename T> __device__ inline T from_f32(float v);
template <> __device__ inline float from_f32<float>(float v) { return v; }
template <> __device__ inline __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

// ---- workspace layout (all offsets 256-byte aligned) --------------------------------------------
// Rotation tables, built on the device in fp64 and stored as fp32 (cos, sin) pairs:
//   key table  T[k][i] = (cos, sin)(Delta(k) * theta_i), k in [0, L), i in [0, d/2)   (SIMT prefill)
//   two-level  HI[a][i] = cs(-(256 a) theta_i), LO[b][i] = cs(-b theta_i), b in [0,256) (decode, UMMA)
// Remote map of the correction rotation.  Aliasing (the paper's default, Eq.(3),(5)): pair i turns by Delta(x) theta_i with
// the integer Delta(x) = floor(x/G) - x.  Frequency interpolation (R17): pair i
// turns by -x phi_i, phi_i = theta_i (1 - gamma_i)(1 - 1/G), gamma_i the NTK-by-parts ramp over r_i = w_pre theta_i / 2 pi.
// The kernels take the second form as "G = 2^30": then floor(x/G) = 0, n = -Delta = x grows by one per key, and the tables
// are built with phi_i in place of theta_i.
struct FreqMap {
    int interp;               // 0: aliasing, 1: frequency interpolation
    double one_minus_inv_G;   // 1 - 1/G (interp only)
    double w_pre, alpha, beta;
};
inline FreqMap alias_map() { return FreqMap{0, 0.0, 0.0, 1.0, 32.0}; }
constexpr long long kInterpG = 1ll << 30;

struct TableHeader {          // first 256 bytes of a table region; lets decode skip a rebuild
    unsigned long long magic;
    double theta;
    long long n_hi;
    int d;
    unsigned check;           // hash of LO[1][*] and HI[n_hi-1][*]: a header whose body was overwritten does not verify
    unsigned gen;             // incremented by every rebuild: a reader that loaded entries early re-reads them if it moved
    int interp;               // the FreqMap the table was built for
    double omg, w_pre, alpha, beta;
};

constexpr unsigned long long kTableMagic = 0x4a45544c4f4e4732ull;  // "JETLONG2": header of a sealed two-level table

constexpr size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

// prefill (SIMT): key table
int build_key_table(float2* tab, long long L, long long G, int d, double theta, cudaStream_t st, FreqMap fm = alias_map());
// decode / UMMA prefill: two-level table; returns bytes via two_level_bytes
size_t two_level_bytes(long long L, int d);
int build_two_level(void* region, long long L, int d, double theta, cudaStream_t st, FreqMap fm = alias_map());

// multiprocessor count of the current device (cached per device)
int sm_count();

// kernels' host launchers (defined in the respective .cu files)
int launch_prefill_simt(const void* Q, const void* K, const void* V, void* out, float* lse, long long L, int H_q,
                        int H_kv, int d, long long w0, long long G, const float2* key_table, int dtype, bool bifocal,
                        cudaStream_t st);
size_t decode_workspace_bytes(long long L, int H_q, int H_kv, int d);
int launch_decode(const void* q, const void* K, const void* V, void* out, float* lse, long long L, int H_q, int H_kv,
                  int d, long long w0, long long G, double theta, int dtype, bool bifocal, void* ws, size_t ws_bytes,
                  cudaStream_t st, FreqMap fm = alias_map());

}  // namespace jetlong
