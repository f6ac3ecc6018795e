// tables.cu -- rotation tables for the correction rotation of Eq.(5)-(6).
//
// Angles Delta(k)*theta_i reach ~1e5 rad at L=128K, so forming them in fp32 is wrong by ~6e-3 rad.
// Every table entry is therefore computed in fp64 on the device (theta_i = rope_theta^(-2i/d) by pow,
// angle = integer * theta_i, sincos in double) and rounded once to fp32.
#include <math.h>

#include "common.cuh"

namespace jetlong {

// frequency of pair i under the remote map: theta_i (aliasing) or phi_i = theta_i (1 - gamma_i)(1 - 1/G) (R17)
__device__ __forceinline__ double map_freq(int i, int d, double log2_theta, const FreqMap& fm) {
    const double th = exp2(-2.0 * (double)i / (double)d * log2_theta);
    if (!fm.interp) return th;
    const double r = fm.w_pre * th / 6.283185307179586476925286766559;
    double gam = (r - fm.alpha) / (fm.beta - fm.alpha);
    gam = gam < 0.0 ? 0.0 : (gam > 1.0 ? 1.0 : gam);
    return th * (1.0 - gam) * fm.one_minus_inv_G;
}

// ---- per-key table: T[k][i] = (cos, sin)(Delta(k) theta_i) ------------------------------------------
__global__ void key_table_kernel(float2* __restrict__ tab, long long L, long long G, int half, double log2_theta,
                                 int d, FreqMap fm) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= L * half) return;
    long long k = idx / half;
    int i = (int)(idx - k * half);
    double th = map_freq(i, d, log2_theta, fm);
    double a = (double)delta_pos(k, G) * th;                       // interpolation: G = 2^30, Delta(k) = -k
    double s, c;
    sincos(a, &s, &c);
    tab[idx] = make_float2((float)c, (float)s);
}

int build_key_table(float2* tab, long long L, long long G, int d, double theta, cudaStream_t st, FreqMap fm) {
    int half = d / 2;
    long long n = L * half;
    int threads = 256;
    long long blocks = (n + threads - 1) / threads;
    key_table_kernel<<<(unsigned)blocks, threads, 0, st>>>(tab, L, fm.interp ? kInterpG : G, half, log2(theta), d, fm);
    note_launch();
    return check_launch("key_table_kernel");
}

// ---- two-level table -----------------------------------------------------------------------------------
// For n = -Delta >= 0 written as n = 256 a + b:  R(Delta) = R(-256 a) R(-b).
//   HI[a][i] = (cos, sin)(-256 a theta_i), a in [0, n_hi)      LO[b][i] = (cos, sin)(-b theta_i), b in [0, 256)
// Independent of G; depends on L only through n_hi = ceil(L/256)+1, so consecutive decode steps skip the
// rebuild (header match) except once every 256 tokens.
// Region layout: [TableHeader (256 B)] [LO: 256*half float2] [HI: n_hi*half float2]
static constexpr unsigned long long kMagic = kTableMagic;

int sm_count() {
    static int cached[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 148; }
    if (cached[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) { cudaGetLastError(); n = 148; }
        cached[dev] = n;
    }
    return cached[dev];
}

size_t two_level_bytes(long long L, int d) {
    long long n_hi = (L + 255) / 256 + 1;
    return 256 + align256((size_t)(256 + n_hi) * (d / 2) * sizeof(float2));
}

// hash of the 2 x 64 float2 entries of LO[1] and HI[n_hi-1] (the first row that is not all (1, 0) and the last row)
__device__ __forceinline__ unsigned table_check(const float2* lo, const float2* hi, long long n_hi, int half, unsigned* red) {
    const int t = threadIdx.x;
    unsigned h = 0;
    if (t < 2 * half) {
        const float2 v = t < half ? lo[half + t] : hi[(n_hi - 1) * half + (t - half)];
        h = (__float_as_uint(v.x) * 0x9E3779B1u) ^ (__float_as_uint(v.y) * 0x85EBCA77u) ^ ((unsigned)t * 0xC2B2AE3Du);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) h ^= __shfl_xor_sync(0xffffffffu, h, o);
    if ((t & 31) == 0) red[t >> 5] = h;
    __syncthreads();
    unsigned r = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) r ^= red[w];
    __syncthreads();
    return r | 1u;                                                    // never 0
}

// One CTA.  Every call launches it; when the header describes (theta, n_hi, d) AND the table verifies against the
// header's check word it returns at once (decode steps 1..n); otherwise it un-seals the header, rebuilds the table
// and seals it again with a new generation number.  The workspace must have been zero-filled before its first use
// (include/jetlong.h), so an unsealed region never carries the magic by accident.
__global__ void __launch_bounds__(1024) two_level_kernel(unsigned char* __restrict__ region, long long n_hi, int half,
                                                         double theta, double log2_theta, int d, FreqMap fm) {
    __shared__ unsigned red[32];
    // Launched with programmatic stream serialization itself: the CTA may become resident while the previous kernel on the
    // stream (the previous decode step's merge, or any caller kernel) drains.  It first waits for that kernel to complete
    // -- so everything the caller enqueued before this call is visible to us AND to our dependents -- and only then lets
    // the programmatically launched consumer (the decode scan) start.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    TableHeader* hdr = reinterpret_cast<TableHeader*>(region);
    float2* lo = reinterpret_cast<float2*>(region + 256);
    float2* hi = lo + 256 * half;
    const bool same_map = hdr->interp == fm.interp && (!fm.interp || (hdr->omg == fm.one_minus_inv_G && hdr->w_pre == fm.w_pre &&
                                                                         hdr->alpha == fm.alpha && hdr->beta == fm.beta));
    const bool sealed = hdr->magic == kMagic && hdr->theta == theta && hdr->n_hi == n_hi && hdr->d == d && same_map;   // uniform
    if (sealed && table_check(lo, hi, n_hi, half, red) == hdr->check) return;
    const unsigned gen = hdr->gen;
    __syncthreads();
    if (threadIdx.x == 0) { hdr->magic = 0; __threadfence(); }        // un-seal before the body changes
    __syncthreads();
    const long long total = (256 + n_hi) * half;
    for (long long idx = threadIdx.x; idx < total; idx += blockDim.x) {
        const long long row = idx / half;
        const int i = (int)(idx - row * half);
        const double th = map_freq(i, d, log2_theta, fm);
        const double n = row < 256 ? (double)row : 256.0 * (double)(row - 256);
        double s, c;
        sincos(-n * th, &s, &c);
        (row < 256 ? lo : hi)[(row < 256 ? row : row - 256) * half + i] = make_float2((float)c, (float)s);
    }
    __threadfence();
    __syncthreads();
    const unsigned chk = table_check(lo, hi, n_hi, half, red);
    if (threadIdx.x == 0) {
        hdr->theta = theta;
        hdr->n_hi = n_hi;
        hdr->d = d;
        hdr->check = chk;
        hdr->gen = gen + 1u;
        hdr->interp = fm.interp; hdr->omg = fm.one_minus_inv_G; hdr->w_pre = fm.w_pre; hdr->alpha = fm.alpha; hdr->beta = fm.beta;
        __threadfence();
        hdr->magic = kMagic;
    }
}

int build_two_level(void* region, long long L, int d, double theta, cudaStream_t st, FreqMap fm) {
    const long long n_hi = (L + 255) / 256 + 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(1);
    cfg.blockDim = dim3(1024);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, two_level_kernel, (unsigned char*)region, n_hi, d / 2, theta, log2(theta), d, fm);
    note_launch(1);
    return check_launch("two_level_kernel");
}

}  // namespace jetlong
