// rot.cuh -- device helpers shared by the tcgen05 prefill and decode kernels: packed fp32x2 arithmetic, the
// two-level (cos, sin) table lookup and the in-shared-memory correction rotation of K tiles (Eq.(5)-(6) P:101-106).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace jetlong {
namespace dev {

__device__ __forceinline__ float ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float max3(float a, float b, float c) {
    float y;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(a), "f"(b), "f"(c));
    return y;
}
// packed fp32x2 arithmetic (FFMA2 / FADD2 / FMUL2 on sm_100)
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t y;
    asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(lo), "f"(hi));
    return y;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t ffma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t y;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(y) : "l"(a), "l"(b), "l"(c));
    return y;
}
__device__ __forceinline__ uint64_t fadd2(uint64_t a, uint64_t b) {
    uint64_t y;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(y) : "l"(a), "l"(b));
    return y;
}
__device__ __forceinline__ uint64_t fmul2(uint64_t a, uint64_t b) {
    uint64_t y;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(y) : "l"(a), "l"(b));
    return y;
}
__device__ __forceinline__ uint64_t fsub2(uint64_t a, uint64_t b) {
    uint64_t y;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(y) : "l"(a), "l"(b));
    return y;
}
// 2^x for two values on the FMA/ALU pipes (no MUFU): x = n + f, n = round(x), f in [-0.5, 0.5];
// 2^f by a degree-3 minimax polynomial (max relative error 7.5e-5), 2^n by adding n to the exponent field.
// Valid for -126 <= x < 128 after the clamp; used for half of the softmax exponentials so the 16/clk/SM MUFU
// pipe stops being the limiter.
__device__ __forceinline__ void exp2_poly2(uint64_t x2, float& r0, float& r1) {
    float x0, x1;
    unpack2(x2, x0, x1);
    const uint64_t xc = pack2(fmaxf(x0, -126.0f), fmaxf(x1, -126.0f));
    const uint64_t MAG = pack2(12582912.0f, 12582912.0f);              // 1.5 * 2^23: the add rounds x to an integer
    const uint64_t t = fadd2(xc, MAG);
    const uint64_t f = fsub2(xc, fsub2(t, MAG));
    uint64_t pl = ffma2(pack2(5.517165290e-02f, 5.517165290e-02f), f, pack2(2.426111210e-01f, 2.426111210e-01f));
    pl = ffma2(pl, f, pack2(6.932609884e-01f, 6.932609884e-01f));
    pl = ffma2(pl, f, pack2(9.999280737e-01f, 9.999280737e-01f));
    float p0, p1, t0, t1;
    unpack2(pl, p0, p1);
    unpack2(t, t0, t1);
    r0 = __uint_as_float(__float_as_uint(p0) + (__float_as_uint(t0) << 23));
    r1 = __uint_as_float(__float_as_uint(p1) + (__float_as_uint(t1) << 23));
}
__device__ __forceinline__ uint32_t bf16x2(float lo, float hi) {
    uint32_t y;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(y) : "f"(hi), "f"(lo));
    return y;
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// producer side of a named barrier: counts this thread in and goes on (the consumer side is named_bar_sync)
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// (cos, sin)(Delta(pos) theta_i) for 8 consecutive frequencies i = i0 .. i0+7 from the two-level table
// (HI[n >> 8] * LO[n & 255] as complex numbers, n = -Delta(pos) >= 0, Eq.(5))
__device__ __forceinline__ void cs8(const float2* __restrict__ lo, const float2* __restrict__ hi, long long pos,
                                    long long G, int i0, float* cs_c, float* cs_s) {
    const long long n = pos - pos / G;
    const float4* ph = reinterpret_cast<const float4*>(hi + (n >> 8) * 64 + i0);
    const float4* pl = reinterpret_cast<const float4*>(lo + (n & 255) * 64 + i0);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 h = __ldg(ph + j), l = __ldg(pl + j);
        cs_c[2 * j] = h.x * l.x - h.y * l.y;      cs_s[2 * j] = h.y * l.x + h.x * l.y;
        cs_c[2 * j + 1] = h.z * l.z - h.w * l.w;  cs_s[2 * j + 1] = h.w * l.z + h.z * l.w;
    }
}

// rotate 8 pairs: a[4] = bf16 words of channels i0..i0+7, b[4] = their partners i0+64..; fp32 rotation, then
// fp16 hi words (h1, h2) and fp16 lo words (l1, l2) of the residual y - hi.
__device__ __forceinline__ void rot8(const uint32_t* a, const uint32_t* b, const float* cs_c, const float* cs_s,
                                     uint32_t* h1, uint32_t* h2, uint32_t* l1, uint32_t* l2) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float x1l = __uint_as_float(a[j] << 16), x1h = __uint_as_float(a[j] & 0xffff0000u);
        const float x2l = __uint_as_float(b[j] << 16), x2h = __uint_as_float(b[j] & 0xffff0000u);
        const float y1l = x1l * cs_c[2 * j] - x2l * cs_s[2 * j];
        const float y2l = x1l * cs_s[2 * j] + x2l * cs_c[2 * j];
        const float y1h = x1h * cs_c[2 * j + 1] - x2h * cs_s[2 * j + 1];
        const float y2h = x1h * cs_s[2 * j + 1] + x2h * cs_c[2 * j + 1];
        const __half2 a1 = __floats2half2_rn(y1l, y1h), a2 = __floats2half2_rn(y2l, y2h);
        const float2 f1 = __half22float2(a1), f2 = __half22float2(a2);
        const __half2 r1 = __floats2half2_rn(y1l - f1.x, y1h - f1.y), r2 = __floats2half2_rn(y2l - f2.x, y2h - f2.y);
        h1[j] = *reinterpret_cast<const uint32_t*>(&a1);
        h2[j] = *reinterpret_cast<const uint32_t*>(&a2);
        l1[j] = *reinterpret_cast<const uint32_t*>(&r1);
        l2[j] = *reinterpret_cast<const uint32_t*>(&r2);
    }
}

// ---- step a5: correction rotation of 16 ROWS key rows of a K tile, in shared memory ---------------------------
// kh: [2 boxes of KBOX bytes][rows][128 B] SWIZZLE_128B, bf16 in, fp16 hi out (in place); kl: same layout, fp16
// lo out.  Thread t of the 128-thread rotate group owns the 16-byte chunk c = t & 7 (channels 8c..8c+7 of box 0
// and their partners 64+8c.. of box 1, i.e. frequencies 8c..8c+7) of the ROWS consecutive rows ROWS(t>>3)+m.
// (cos, sin) of the first row come from the two-level table, fetched ONE VISIT AHEAD (KRot::prefetch) so no
// global-load latency sits between the TMA arrival and the MMA; rows 1..3 follow by the exact recurrence
// cs(n+1) = cs(n) * cs(1) (n = -Delta grows by 1 per key, by 0 when the key position is a multiple of G);
// the recurrence runs at most 7 steps from a table value, so it adds no measurable error.
// All arithmetic is packed fp32x2 (FFMA2/FMUL2): a bf16 word holds two adjacent channels = two frequencies.
template <int ROWS> struct KRot {
    uint64_t sc[4], ss[4];          // unit step cs(-theta_i), pairs of frequencies (8c+2j, 8c+2j+1)
    float4 nh[4], nl[4];            // prefetched HI / LO table entries of the next visit's first row
    const float2* lo; const float2* hi;
    int c, r0;
    unsigned G;
    unsigned rem_, n_;              // decode (consecutive tiles): position mod G and n of this thread's first row, carried
    __device__ __forceinline__ void init(const float2* lo_, const float2* hi_, int t, long long G_, int rbase = 0) {
        lo = lo_; hi = hi_; c = t & 7; r0 = rbase + ROWS * (t >> 3); G = (unsigned)G_;
        const float4* p1 = reinterpret_cast<const float4*>(lo + 64 + 8 * c);       // LO[1][8c..]
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const float4 l = __ldg(p1 + j);
            sc[j] = pack2(l.x, l.z); ss[j] = pack2(l.y, l.w);
        }
    }
    // the same with the thread's chunk (8 frequency pairs) and first row given by the caller
    __device__ __forceinline__ void init_at(const float2* lo_, const float2* hi_, int c_, int r0_, long long G_) {
        init(lo_, hi_, c_, G_);
        r0 = r0_;
    }
    // carried form for a run of consecutive 128-key tiles: seek() once (two divisions), then step128() per tile (none)
    __device__ __forceinline__ void seek(unsigned pos0) {
        const unsigned pos = pos0 + r0;
        rem_ = pos % G; n_ = pos - pos / G;
    }
    __device__ __forceinline__ void step128(unsigned m128, unsigned d128) {        // m128 = 128 % G, d128 = 128 / G
        rem_ += m128;
        const unsigned wrap = rem_ >= G ? 1u : 0u;
        rem_ -= wrap ? G : 0u;
        n_ += 128u - d128 - wrap;
    }
    __device__ __forceinline__ void prefetch_carried() {
        const float4* ph = reinterpret_cast<const float4*>(hi + (size_t)(n_ >> 8) * 64 + 8 * c);
        const float4* pl = reinterpret_cast<const float4*>(lo + (size_t)(n_ & 255) * 64 + 8 * c);
#pragma unroll
        for (int j = 0; j < 4; ++j) { nh[j] = __ldg(ph + j); nl[j] = __ldg(pl + j); }
    }
    // pos0 = absolute position of this CTA's first key row of the tile
    __device__ __forceinline__ void prefetch(unsigned pos0) {
        const unsigned pos = pos0 + r0;
        const unsigned n = pos - pos / G;
        const float4* ph = reinterpret_cast<const float4*>(hi + (size_t)(n >> 8) * 64 + 8 * c);
        const float4* pl = reinterpret_cast<const float4*>(lo + (size_t)(n & 255) * 64 + 8 * c);
#pragma unroll
        for (int j = 0; j < 4; ++j) { nh[j] = __ldg(ph + j); nl[j] = __ldg(pl + j); }
    }
};

__device__ __forceinline__ uint64_t neg2(uint64_t v) { return v ^ 0x8000000080000000ull; }
// both halves on the ALU pipe (PRMT, LOP3): ptxas turns `w << 16` into IMAD.SHL, which competes with the rotation's
// FFMA2/FMUL2 for the FMA pipe -- the pipe that bounds the rotate group (measured)
__device__ __forceinline__ uint64_t bf16x2_to_f32x2(uint32_t w) {
    return (uint64_t)__byte_perm(w, 0u, 0x1044) | ((uint64_t)(w & 0xffff0000u) << 32);
}
__device__ __forceinline__ uint32_t f16x2_rn(float lo, float hi) {
    uint32_t y;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(y) : "f"(hi), "f"(lo));
    return y;
}
// y (packed f32x2) -> fp16x2 hi word and fp16x2 word of the residual y - hi
__device__ __forceinline__ void split_hi_lo(uint64_t y, uint32_t& h, uint32_t& l, bool precise) {
    float a, b;
    unpack2(y, a, b);
    h = f16x2_rn(a, b);
    if (precise) {
        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&h));
        float ra, rb;
        unpack2(fsub2(y, pack2(f.x, f.y)), ra, rb);                   // one packed subtract for the two residuals
        l = f16x2_rn(ra, rb);
    }
}

// four e5m2 bytes from two fp16x2 words: e5m2 is the top byte of fp16 (same exponent bias); +0x80 rounds to nearest
__device__ __forceinline__ uint32_t e5m2x4(uint32_t w0, uint32_t w1) {
    return __byte_perm(w0 + 0x00800080u, w1 + 0x00800080u, 0x7531);
}
__device__ __forceinline__ void sts16s(uint32_t a, uint32_t v) {           // low 16 bits of v
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v) : "memory");
}
__device__ __forceinline__ void sts64(uint32_t a, uint32_t x, uint32_t y) {
    asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(a), "r"(x), "r"(y) : "memory");
}

// explicit shared-space 128-bit accesses (pointers that pass through lambdas degrade to generic LD/ST otherwise)
__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

template <int ROWS, int KBOX>
__device__ __forceinline__ void rotate_k_rows(uint32_t kh, uint32_t kl, unsigned pos0, KRot<ROWS>& R, int precise) {   // kh, kl: shared-space addresses
    // precise: 0 = hi only; 1 = fp16 lo at kl (same layout as kh); 2 = e5m2 copies for the cross terms at kl:
    //          [box of KBOX bytes: K' as e5m2, rows x 128 channels][box: K' lo as e5m2], SWIZZLE_128B;
    //          3 = only K' lo as e5m2 at kl (one box)
    // first-row (cos, sin) from the prefetched table entries: HI * LO as complex numbers
    uint64_t cc[4], cs[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 h = R.nh[j], l = R.nl[j];
        cc[j] = pack2(h.x * l.x - h.y * l.y, h.z * l.z - h.w * l.w);
        cs[j] = pack2(h.y * l.x + h.x * l.y, h.w * l.z + h.z * l.w);
    }
    unsigned rem = (pos0 + R.r0) % R.G;
#pragma unroll
    for (int m = 0; m < ROWS; ++m) {
        const int r = R.r0 + m;
        if (m > 0) {
            rem = (rem + 1 == R.G) ? 0u : rem + 1;
            if (rem != 0) {                                           // n grows by one: advance by the unit step
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint64_t c2 = ffma2(neg2(cs[j]), R.ss[j], fmul2(cc[j], R.sc[j]));
                    cs[j] = ffma2(cc[j], R.ss[j], fmul2(cs[j], R.sc[j]));
                    cc[j] = c2;
                }
            }
        }
        const int off = r * 128 + ((R.c ^ (r & 7)) << 4);
        const uint4 u1 = lds128(kh + off);
        const uint4 u2 = lds128(kh + KBOX + off);
        const uint32_t a[4] = {u1.x, u1.y, u1.z, u1.w}, b[4] = {u2.x, u2.y, u2.z, u2.w};
        uint32_t h1[4], h2[4], l1[4], l2[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint64_t x1 = bf16x2_to_f32x2(a[j]), x2 = bf16x2_to_f32x2(b[j]);
            const uint64_t y1 = ffma2(neg2(x2), cs[j], fmul2(x1, cc[j]));      // x1 c - x2 s
            const uint64_t y2 = ffma2(x1, cs[j], fmul2(x2, cc[j]));            // x1 s + x2 c
            split_hi_lo(y1, h1[j], l1[j], precise != 0);
            split_hi_lo(y2, h2[j], l2[j], precise != 0);
        }
        sts128(kh + off, h1[0], h1[1], h1[2], h1[3]);
        sts128(kh + KBOX + off, h2[0], h2[1], h2[2], h2[3]);
        if (precise == 1) {
            sts128(kl + off, l1[0], l1[1], l1[2], l1[3]);
            sts128(kl + KBOX + off, l2[0], l2[1], l2[2], l2[3]);
        } else if (precise == 2) {
            // byte b of an e5m2 row is channel b: channels 8c.. sit in 16-byte chunk c/2, channels 64+8c.. in chunk 4+c/2
            const uint32_t o1 = r * 128 + ((((R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            const uint32_t o2 = r * 128 + (((4 + (R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            const uint32_t a0 = e5m2x4(h1[0], h1[1]), a1 = e5m2x4(h1[2], h1[3]), b0 = e5m2x4(h2[0], h2[1]), b1 = e5m2x4(h2[2], h2[3]);
            const uint32_t c0 = e5m2x4(l1[0], l1[1]), c1 = e5m2x4(l1[2], l1[3]), d0 = e5m2x4(l2[0], l2[1]), d1 = e5m2x4(l2[2], l2[3]);
            sts64(kl + o1, a0, a1);
            sts64(kl + o2, b0, b1);
            sts64(kl + KBOX + o1, c0, c1);
            sts64(kl + KBOX + o2, d0, d1);
        } else if (precise == 3) {
            const uint32_t o1 = r * 128 + ((((R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            const uint32_t o2 = r * 128 + (((4 + (R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            sts64(kl + o1, e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3]));
            sts64(kl + o2, e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]));
        }
    }
}

// ---- lean form of the correction rotation (two-tile prefill) ---------------------------------------------------
// Same arithmetic as rotate_k_rows, about half the instructions per key row (measured with ncu: 250 -> ~125):
//   * (cos, sin, -sin) are all carried, so neither the rotation nor the recurrence negates a packed operand per use;
//   * the residual is one mixed-precision FHADD per value (sub.f32.f16: hi - y = -lo) instead of two conversions and a
//     packed subtract; the consumer undoes the sign with the negate bit of the UMMA instruction descriptor;
//   * MODE 5 (selective compensation): the two selected pairs of the chunk are picked from the fp16 words with a
//     three-PRMT tree BEFORE the e5m2 rounding, and each thread stores one 32-bit word per region:
//       compact row = region LO at byte b_lo: 8 chunks x [lo1(f0) lo1(f1) lo2(f0) lo2(f1)], region HI at b_hi: the same of hi
//     (position j of the 32-byte contraction slice means the same (chunk, pair, half) in Q' and K' rows, which is all the
//     UMMA needs);
//   * the next row's shared-memory loads are issued before the current row's arithmetic.
// MODE 0: hi only.  MODE 2: full e5m2 copies at kl (as rotate_k_rows mode 2, lo negated).  MODE 3: only -lo as e5m2 at kl
// (decode).  MODE 5 as above.  MODE 6: as 5 with fp16 instead of e5m2 (regions of 64 bytes).
__device__ __forceinline__ float fhsub_lo(uint32_t h, float y) {     // (low fp16 of h) - y
    float r;
    unsigned short hs;
    asm("{.reg .b16 t; mov.b32 {%0, t}, %1;}" : "=h"(hs) : "r"(h));
    asm("sub.rn.f32.f16 %0, %1, %2;" : "=f"(r) : "h"(hs), "f"(y));
    return r;
}
__device__ __forceinline__ float fhsub_hi(uint32_t h, float y) {     // (high fp16 of h) - y
    float r;
    unsigned short hs;
    asm("{.reg .b16 t; mov.b32 {t, %0}, %1;}" : "=h"(hs) : "r"(h));
    asm("sub.rn.f32.f16 %0, %1, %2;" : "=f"(r) : "h"(hs), "f"(y));
    return r;
}
// selectors of the PRMT tree for the two compensated pairs f0 < f1 (0..7) of a chunk, from selw = f0 | f1 << 4
struct SelTree {
    uint32_t s_pool, s_top;
    __device__ __forceinline__ void init(uint32_t selw) {
        const uint32_t f0 = selw & 7u, f1 = (selw >> 4) & 7u;
        const uint32_t h0 = 2u * (f0 & 3u), h1 = 2u * (f1 & 3u);
        s_pool = h0 | ((h0 + 1u) << 4) | (h1 << 8) | ((h1 + 1u) << 12);           // the same selector serves both pools
        const uint32_t a = f0 < 4u ? 0u : 4u, b = f1 < 4u ? 2u : 6u;
        s_top = a | ((a + 1u) << 4) | (b << 8) | ((b + 1u) << 12);
    }
    // [half f0 | half f1] of the eight fp16 halves in w[0..3]
    __device__ __forceinline__ uint32_t pick(const uint32_t (&w)[4]) const {
        return __byte_perm(__byte_perm(w[0], w[1], s_pool), __byte_perm(w[2], w[3], s_pool), s_top);
    }
};

template <int ROWS, int KBOX, int MODE, bool UNROLL = false, bool CARRIED = false, int RR = ROWS>
__device__ __forceinline__ void rotate_rows2(uint32_t kh, uint32_t kl, unsigned pos0, KRot<RR>& R, const SelTree& T,
                                             uint32_t b_lo, uint32_t b_hi) {
    uint64_t cc[4], cs[4], ncs[4], nss[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 h = R.nh[j], l = R.nl[j];
        cc[j] = pack2(h.x * l.x - h.y * l.y, h.z * l.z - h.w * l.w);
        cs[j] = pack2(h.y * l.x + h.x * l.y, h.w * l.z + h.z * l.w);
        ncs[j] = neg2(cs[j]);
        nss[j] = neg2(R.ss[j]);
    }
    unsigned rem = CARRIED ? R.rem_ : (pos0 + R.r0) % R.G;              // CARRIED: the caller keeps it (KRot::seek / step128)
    int off = R.r0 * 128 + ((R.c ^ (R.r0 & 7)) << 4);
    uint4 u1 = lds128(kh + off), u2 = lds128(kh + KBOX + off);
    // rolled on purpose: the SM's instruction caches are small (L0 ~6 KB, L1.5 32 KB) and four roles run different loops;
    // unrolled, this loop alone was 16 KB and its warps spent most samples in stall_no_inst (ncu)
#pragma unroll(UNROLL ? ROWS : 1)
    for (int m = 0; m < ROWS; ++m) {
        const int r = R.r0 + m;
        const int off_n = (r + 1) * 128 + ((R.c ^ ((r + 1) & 7)) << 4);
        uint4 n1 = u1, n2 = u2;
        if (m + 1 < ROWS) { n1 = lds128(kh + off_n); n2 = lds128(kh + KBOX + off_n); }
        const uint32_t a[4] = {u1.x, u1.y, u1.z, u1.w}, b[4] = {u2.x, u2.y, u2.z, u2.w};
        uint32_t h1[4], h2[4], l1[4], l2[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint64_t x1 = bf16x2_to_f32x2(a[j]), x2 = bf16x2_to_f32x2(b[j]);
            const uint64_t y1 = ffma2(x2, ncs[j], fmul2(x1, cc[j]));           // x1 c - x2 s
            const uint64_t y2 = ffma2(x1, cs[j], fmul2(x2, cc[j]));            // x1 s + x2 c
            float y1a, y1b, y2a, y2b;
            unpack2(y1, y1a, y1b);
            unpack2(y2, y2a, y2b);
            h1[j] = f16x2_rn(y1a, y1b);
            h2[j] = f16x2_rn(y2a, y2b);
            if (MODE != 0) {                                                   // -lo = hi - y
                l1[j] = f16x2_rn(fhsub_lo(h1[j], y1a), fhsub_hi(h1[j], y1b));
                l2[j] = f16x2_rn(fhsub_lo(h2[j], y2a), fhsub_hi(h2[j], y2b));
            }
        }
        sts128(kh + off, h1[0], h1[1], h1[2], h1[3]);
        sts128(kh + KBOX + off, h2[0], h2[1], h2[2], h2[3]);
        if (MODE == 2) {
            // byte b of an e5m2 row is channel b: channels 8c.. sit in 16-byte chunk c/2, channels 64+8c.. in chunk 4+c/2
            const uint32_t o1 = r * 128 + ((((R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            const uint32_t o2 = r * 128 + (((4 + (R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            sts64(kl + o1, e5m2x4(h1[0], h1[1]), e5m2x4(h1[2], h1[3]));
            sts64(kl + o2, e5m2x4(h2[0], h2[1]), e5m2x4(h2[2], h2[3]));
            sts64(kl + KBOX + o1, e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3]));
            sts64(kl + KBOX + o2, e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]));
        } else if (MODE == 3) {                                        // decode: only K' lo as e5m2 at kl (one box)
            const uint32_t o1 = r * 128 + ((((R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            const uint32_t o2 = r * 128 + (((4 + (R.c >> 1)) ^ (r & 7)) << 4) + (R.c & 1) * 8;
            sts64(kl + o1, e5m2x4(l1[0], l1[1]), e5m2x4(l1[2], l1[3]));
            sts64(kl + o2, e5m2x4(l2[0], l2[1]), e5m2x4(l2[2], l2[3]));
        } else if (MODE == 5) {
            const uint32_t x = (uint32_t)(r & 7), cw = (uint32_t)(R.c >> 2), cb = (uint32_t)(R.c & 3) * 4u;
            const uint32_t wl = __byte_perm(T.pick(l1) + 0x00800080u, T.pick(l2) + 0x00800080u, 0x7531);
            const uint32_t wh = __byte_perm(T.pick(h1) + 0x00800080u, T.pick(h2) + 0x00800080u, 0x7531);
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(kl + r * 128 + ((((b_lo >> 4) + cw) ^ x) << 4) + cb), "r"(wl) : "memory");
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(kl + r * 128 + ((((b_hi >> 4) + cw) ^ x) << 4) + cb), "r"(wh) : "memory");
        } else if (MODE == 6) {
            // MODE 5 with the selected pairs kept in fp16: regions of 64 bytes, chunk c = 8 bytes [x1(f0) x1(f1) | x2(f0) x2(f1)]
            const uint32_t x = (uint32_t)(r & 7), cw = (uint32_t)(R.c >> 1), cb = (uint32_t)(R.c & 1) * 8u;
            sts64(kl + r * 128 + ((((b_lo >> 4) + cw) ^ x) << 4) + cb, T.pick(l1), T.pick(l2));
            sts64(kl + r * 128 + ((((b_hi >> 4) + cw) ^ x) << 4) + cb, T.pick(h1), T.pick(h2));
        }
        if (m + 1 < ROWS) {
            rem = (rem + 1 == R.G) ? 0u : rem + 1;
            if (rem != 0) {                                           // n grows by one: advance by the unit step
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint64_t c2 = ffma2(cs[j], nss[j], fmul2(cc[j], R.sc[j]));
                    cs[j] = ffma2(cc[j], R.ss[j], fmul2(cs[j], R.sc[j]));
                    cc[j] = c2;
                    ncs[j] = neg2(cs[j]);
                }
            }
        }
        off = off_n; u1 = n1; u2 = n2;
    }
}

}  // namespace dev
}  // namespace jetlong
