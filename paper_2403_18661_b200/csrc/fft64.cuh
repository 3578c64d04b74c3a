// Register-resident 64-point complex DFT (8 x 8 Cooley-Tukey, fully unrolled, every index a compile-time constant) and
// the pieces of the 4096-point = 64 x 64 two-pass transform built on it (signal_fft64.cu).
//
// Why this shape (profiles/r01d_whiten_full.md): the round-1 kernels ran a 4096-point transform as
// three radix-16 Stockham passes through shared memory with 256 threads.  They were bound by instruction issue AND by
// shared-memory bandwidth: 128 B of shared-memory traffic per complex element and transform pair, 14 block-wide
// barriers, a 14-multiply twiddle product tree per thread and pass, and a separate untangle loop.  With 64 elements per
// thread a 4096-point transform needs TWO passes: one trip through shared memory between them (16 B per element), the
// first pass reads global memory and the last one writes it, twiddles come from a [64][64] shared-memory table
// (conflict-free, one LDS per element), and 64 independent butterflies per thread hide every latency without
// occupancy.
#pragma once
#include "common.cuh"

// (cos, sin)(2 pi m / 64), rounded once from double
__device__ __forceinline__ float2 w64_cs(int m) {
  switch (m & 63) {
    case 0: return make_float2(1.0f, 0.0f);
    case 1: return make_float2(0.9951847266721969f, 0.0980171403295606f);
    case 2: return make_float2(0.9807852804032304f, 0.19509032201612825f);
    case 3: return make_float2(0.9569403357322088f, 0.29028467725446233f);
    case 4: return make_float2(0.9238795325112867f, 0.3826834323650898f);
    case 5: return make_float2(0.881921264348355f, 0.47139673682599764f);
    case 6: return make_float2(0.8314696123025452f, 0.5555702330196022f);
    case 7: return make_float2(0.773010453362737f, 0.6343932841636455f);
    case 8: return make_float2(0.7071067811865476f, 0.7071067811865475f);
    case 9: return make_float2(0.6343932841636455f, 0.773010453362737f);
    case 10: return make_float2(0.5555702330196023f, 0.8314696123025452f);
    case 11: return make_float2(0.4713967368259978f, 0.8819212643483549f);
    case 12: return make_float2(0.38268343236508984f, 0.9238795325112867f);
    case 13: return make_float2(0.29028467725446233f, 0.9569403357322089f);
    case 14: return make_float2(0.19509032201612833f, 0.9807852804032304f);
    case 15: return make_float2(0.09801714032956077f, 0.9951847266721968f);
    case 16: return make_float2(6.123233995736766e-17f, 1.0f);
    case 17: return make_float2(-0.09801714032956065f, 0.9951847266721969f);
    case 18: return make_float2(-0.1950903220161282f, 0.9807852804032304f);
    case 19: return make_float2(-0.29028467725446216f, 0.9569403357322089f);
    case 20: return make_float2(-0.3826834323650897f, 0.9238795325112867f);
    case 21: return make_float2(-0.4713967368259977f, 0.881921264348355f);
    case 22: return make_float2(-0.555570233019602f, 0.8314696123025455f);
    case 23: return make_float2(-0.6343932841636454f, 0.7730104533627371f);
    case 24: return make_float2(-0.7071067811865475f, 0.7071067811865476f);
    case 25: return make_float2(-0.773010453362737f, 0.6343932841636455f);
    case 26: return make_float2(-0.8314696123025453f, 0.5555702330196022f);
    case 27: return make_float2(-0.8819212643483549f, 0.47139673682599786f);
    case 28: return make_float2(-0.9238795325112867f, 0.3826834323650899f);
    case 29: return make_float2(-0.9569403357322088f, 0.2902846772544624f);
    case 30: return make_float2(-0.9807852804032304f, 0.1950903220161286f);
    case 31: return make_float2(-0.9951847266721968f, 0.09801714032956083f);
    case 32: return make_float2(-1.0f, 1.2246467991473532e-16f);
    case 33: return make_float2(-0.9951847266721969f, -0.09801714032956059f);
    case 34: return make_float2(-0.9807852804032304f, -0.19509032201612836f);
    case 35: return make_float2(-0.9569403357322089f, -0.2902846772544621f);
    case 36: return make_float2(-0.9238795325112868f, -0.38268343236508967f);
    case 37: return make_float2(-0.881921264348355f, -0.47139673682599764f);
    case 38: return make_float2(-0.8314696123025455f, -0.555570233019602f);
    case 39: return make_float2(-0.7730104533627371f, -0.6343932841636453f);
    case 40: return make_float2(-0.7071067811865477f, -0.7071067811865475f);
    case 41: return make_float2(-0.6343932841636459f, -0.7730104533627367f);
    case 42: return make_float2(-0.5555702330196022f, -0.8314696123025452f);
    case 43: return make_float2(-0.47139673682599786f, -0.8819212643483549f);
    case 44: return make_float2(-0.38268343236509034f, -0.9238795325112865f);
    case 45: return make_float2(-0.29028467725446244f, -0.9569403357322088f);
    case 46: return make_float2(-0.19509032201612866f, -0.9807852804032303f);
    case 47: return make_float2(-0.09801714032956045f, -0.9951847266721969f);
    case 48: return make_float2(-1.8369701987210297e-16f, -1.0f);
    case 49: return make_float2(0.09801714032956009f, -0.9951847266721969f);
    case 50: return make_float2(0.1950903220161283f, -0.9807852804032304f);
    case 51: return make_float2(0.29028467725446205f, -0.9569403357322089f);
    case 52: return make_float2(0.38268343236509f, -0.9238795325112866f);
    case 53: return make_float2(0.4713967368259976f, -0.881921264348355f);
    case 54: return make_float2(0.5555702330196018f, -0.8314696123025455f);
    case 55: return make_float2(0.6343932841636456f, -0.7730104533627369f);
    case 56: return make_float2(0.7071067811865474f, -0.7071067811865477f);
    case 57: return make_float2(0.7730104533627367f, -0.6343932841636459f);
    case 58: return make_float2(0.8314696123025452f, -0.5555702330196022f);
    case 59: return make_float2(0.8819212643483548f, -0.4713967368259979f);
    case 60: return make_float2(0.9238795325112865f, -0.3826834323650904f);
    case 61: return make_float2(0.9569403357322088f, -0.2902846772544625f);
    case 62: return make_float2(0.9807852804032303f, -0.19509032201612872f);
    case 63: return make_float2(0.9951847266721969f, -0.0980171403295605f);
  }
  return make_float2(1.f, 0.f);
}

// (cos, sin)(2 pi m / 128), m < 32
__device__ __forceinline__ float2 w128_cs(int m) {
  switch (m & 31) {
    case 0: return make_float2(1.0f, 0.0f);
    case 1: return make_float2(0.9987954562051724f, 0.049067674327418015f);
    case 2: return make_float2(0.9951847266721969f, 0.0980171403295606f);
    case 3: return make_float2(0.989176509964781f, 0.14673047445536175f);
    case 4: return make_float2(0.9807852804032304f, 0.19509032201612825f);
    case 5: return make_float2(0.970031253194544f, 0.24298017990326387f);
    case 6: return make_float2(0.9569403357322088f, 0.29028467725446233f);
    case 7: return make_float2(0.9415440651830208f, 0.33688985339222005f);
    case 8: return make_float2(0.9238795325112867f, 0.3826834323650898f);
    case 9: return make_float2(0.9039892931234433f, 0.4275550934302821f);
    case 10: return make_float2(0.881921264348355f, 0.47139673682599764f);
    case 11: return make_float2(0.8577286100002721f, 0.5141027441932217f);
    case 12: return make_float2(0.8314696123025452f, 0.5555702330196022f);
    case 13: return make_float2(0.8032075314806449f, 0.5956993044924334f);
    case 14: return make_float2(0.773010453362737f, 0.6343932841636455f);
    case 15: return make_float2(0.7409511253549591f, 0.6715589548470183f);
    case 16: return make_float2(0.7071067811865476f, 0.7071067811865475f);
    case 17: return make_float2(0.6715589548470183f, 0.7409511253549591f);
    case 18: return make_float2(0.6343932841636455f, 0.773010453362737f);
    case 19: return make_float2(0.5956993044924335f, 0.8032075314806448f);
    case 20: return make_float2(0.5555702330196023f, 0.8314696123025452f);
    case 21: return make_float2(0.5141027441932217f, 0.8577286100002721f);
    case 22: return make_float2(0.4713967368259978f, 0.8819212643483549f);
    case 23: return make_float2(0.4275550934302822f, 0.9039892931234433f);
    case 24: return make_float2(0.38268343236508984f, 0.9238795325112867f);
    case 25: return make_float2(0.33688985339222005f, 0.9415440651830208f);
    case 26: return make_float2(0.29028467725446233f, 0.9569403357322089f);
    case 27: return make_float2(0.24298017990326398f, 0.970031253194544f);
    case 28: return make_float2(0.19509032201612833f, 0.9807852804032304f);
    case 29: return make_float2(0.14673047445536175f, 0.989176509964781f);
    case 30: return make_float2(0.09801714032956077f, 0.9951847266721968f);
    case 31: return make_float2(0.049067674327418126f, 0.9987954562051724f);
  }
  return make_float2(1.f, 0.f);
}

// a * (S i): S = -1 forward transforms (W_N = exp(-2 pi i / N)), S = +1 inverse (unnormalised)
template <int S> __device__ __forceinline__ float2 f64_mul_i(float2 a) {
  return S < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}
__device__ __forceinline__ float2 f64_add(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 f64_sub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// a * (c + i S s), c and s compile-time constants after unrolling
template <int S> __device__ __forceinline__ float2 f64_cmul_cs(float2 a, float2 cs) {
  const float s = S < 0 ? -cs.y : cs.y;
  return make_float2(fmaf(a.x, cs.x, -(a.y * s)), fmaf(a.y, cs.x, a.x * s));
}
// a * w, w a run-time value; CONJ: a * conj(w)
template <bool CONJ> __device__ __forceinline__ float2 f64_cmul(float2 a, float2 w) {
  if (CONJ) return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(a.y, w.x, -(a.x * w.y)));
  return make_float2(fmaf(a.x, w.x, -(a.y * w.y)), fmaf(a.y, w.x, a.x * w.y));
}

// 4-point DFT, natural order in and out
template <int S> __device__ __forceinline__ void fft4(float2& a, float2& b, float2& c, float2& d) {
  const float2 t0 = f64_add(a, c), t1 = f64_sub(a, c), t2 = f64_add(b, d), t3 = f64_mul_i<S>(f64_sub(b, d));
  a = f64_add(t0, t2); c = f64_sub(t0, t2); b = f64_add(t1, t3); d = f64_sub(t1, t3);
}

// 8-point DFT, natural order in and out (radix-2 decimation in time over two 4-point DFTs; 52 instructions)
template <int S>
__device__ __forceinline__ void fft8(float2& x0, float2& x1, float2& x2, float2& x3, float2& x4, float2& x5, float2& x6, float2& x7) {
  fft4<S>(x0, x2, x4, x6);                       // E0..E3 in x0, x2, x4, x6
  fft4<S>(x1, x3, x5, x7);                       // O0..O3 in x1, x3, x5, x7
  const float h = 0.70710678118654752440f;
  const float2 e0 = x0, e1 = x2, e2 = x4, e3 = x6, o0 = x1, o1 = x3, o2 = x5, o3 = x7;
  // W8^1 = (1 + S i) / sqrt 2, W8^2 = S i, W8^3 = (-1 + S i) / sqrt 2
  const float2 t1 = S < 0 ? make_float2(o1.x + o1.y, o1.y - o1.x) : make_float2(o1.x - o1.y, o1.y + o1.x);
  const float2 t2 = f64_mul_i<S>(o2);
  const float2 u3 = S < 0 ? make_float2(o3.x - o3.y, o3.y + o3.x) : make_float2(o3.x + o3.y, o3.y - o3.x);   // = -sqrt2 W8^3 o3
  x0 = f64_add(e0, o0); x4 = f64_sub(e0, o0);
  x1 = make_float2(fmaf(h, t1.x, e1.x), fmaf(h, t1.y, e1.y)); x5 = make_float2(fmaf(-h, t1.x, e1.x), fmaf(-h, t1.y, e1.y));
  x2 = f64_add(e2, t2); x6 = f64_sub(e2, t2);
  x3 = make_float2(fmaf(-h, u3.x, e3.x), fmaf(-h, u3.y, e3.y)); x7 = make_float2(fmaf(h, u3.x, e3.x), fmaf(h, u3.y, e3.y));
}

// Eight 8-point DFTs side by side: transform l (0..7) takes its element e (0..7) from v[e * ES + l * VS], natural order in
// and out.  Every butterfly level is written ACROSS the eight transforms, so consecutive instructions are independent:
// a warp issues in order, and with 64 elements per thread there are only two warps per scheduler to cover the 4-cycle
// dependent-issue latency (one transform after the other left the issue slots half empty).
template <int S, int ES, int VS> __device__ __forceinline__ void fft8x8(float2 (&v)[64]) {
#define F64_X(e) v[(e) * ES + l * VS]
  // level 1: x0 +- x4, x2 +- x6, x1 +- x5, x3 +- x7 (the differences of the second pairs rotated by S i)
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(0), c = F64_X(4); F64_X(0) = f64_add(a, c); F64_X(4) = f64_sub(a, c); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(1), c = F64_X(5); F64_X(1) = f64_add(a, c); F64_X(5) = f64_sub(a, c); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(2), c = F64_X(6); F64_X(2) = f64_add(a, c); F64_X(6) = f64_mul_i<S>(f64_sub(a, c)); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(3), c = F64_X(7); F64_X(3) = f64_add(a, c); F64_X(7) = f64_mul_i<S>(f64_sub(a, c)); }
  // level 2: E0, E2 <- x0 +- x2; E1, E3 <- x4 +- x6; O0, O2 <- x1 +- x3; O1, O3 <- x5 +- x7
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(0), c = F64_X(2); F64_X(0) = f64_add(a, c); F64_X(2) = f64_sub(a, c); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(4), c = F64_X(6); F64_X(4) = f64_add(a, c); F64_X(6) = f64_sub(a, c); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(1), c = F64_X(3); F64_X(1) = f64_add(a, c); F64_X(3) = f64_sub(a, c); }
#pragma unroll
  for (int l = 0; l < 8; ++l) { const float2 a = F64_X(5), c = F64_X(7); F64_X(5) = f64_add(a, c); F64_X(7) = f64_sub(a, c); }
  // now E0 @0, E1 @4, E2 @2, E3 @6, O0 @1, O1 @5, O2 @3, O3 @7.  Level 3: X[k] = E[k] + W8^k O[k], X[k + 4] = E[k] - W8^k O[k],
  // W8^1 = (1 + S i) / sqrt 2, W8^2 = S i, W8^3 = (-1 + S i) / sqrt 2
  const float h = 0.70710678118654752440f;
#pragma unroll
  for (int l = 0; l < 8; ++l) {
    const float2 e0 = F64_X(0), e1 = F64_X(4), e2 = F64_X(2), e3 = F64_X(6), o0 = F64_X(1), o1 = F64_X(5), o2 = F64_X(3), o3 = F64_X(7);
    const float2 t1 = S < 0 ? make_float2(o1.x + o1.y, o1.y - o1.x) : make_float2(o1.x - o1.y, o1.y + o1.x);
    const float2 t2 = f64_mul_i<S>(o2);
    const float2 u3 = S < 0 ? make_float2(o3.x - o3.y, o3.y + o3.x) : make_float2(o3.x + o3.y, o3.y - o3.x);   // = -sqrt2 W8^3 o3
    F64_X(0) = f64_add(e0, o0); F64_X(4) = f64_sub(e0, o0);
    F64_X(1) = make_float2(fmaf(h, t1.x, e1.x), fmaf(h, t1.y, e1.y)); F64_X(5) = make_float2(fmaf(-h, t1.x, e1.x), fmaf(-h, t1.y, e1.y));
    F64_X(2) = f64_add(e2, t2); F64_X(6) = f64_sub(e2, t2);
    F64_X(3) = make_float2(fmaf(-h, u3.x, e3.x), fmaf(-h, u3.y, e3.y)); F64_X(7) = make_float2(fmaf(h, u3.x, e3.x), fmaf(h, u3.y, e3.y));
  }
#undef F64_X
}

// 64-point DFT of v[0..63], natural order in and out: index n = 8 a + b, k = c + 8 d,
//   X[c + 8 d] = sum_b W8^{b d} [ W64^{b c} sum_a W8^{a c} x[8 a + b] ]
template <int S> __device__ __forceinline__ void fft64(float2 (&v)[64]) {
  fft8x8<S, 8, 1>(v);                            // over a, side by side in b: U[c][b] -> v[8 c + b]
#pragma unroll
  for (int c = 1; c < 8; ++c)
#pragma unroll
    for (int b = 1; b < 8; ++b) {
      const int m = c * b;                       // W64^{S m}
      float2& x = v[8 * c + b];
      if (m % 16 == 0) {                         // quarter turns: exact
        const int q = (m / 16) & 3;
        if (q == 1) x = f64_mul_i<S>(x);
        else if (q == 2) x = make_float2(-x.x, -x.y);
        else if (q == 3) x = f64_mul_i<-S>(x);
      } else {
        x = f64_cmul_cs<S>(x, w64_cs(m));
      }
    }
  fft8x8<S, 1, 8>(v);                            // over b, side by side in c: X[c + 8 d] -> v[8 c + d]
  float2 o[64];
#pragma unroll
  for (int c = 0; c < 8; ++c)
#pragma unroll
    for (int d = 0; d < 8; ++d) o[c + 8 * d] = v[8 * c + d];
#pragma unroll
  for (int k = 0; k < 64; ++k) v[k] = o[k];      // (a renaming: no instructions)
}

// ---- 4096 = 64 x 64 ---------------------------------------------------------------------------------------------------
// One transform is run by 64 threads (thread t), 64 elements each, through a [64][F64_ROW] float2 shared-memory tile
// (rows padded to 65 elements: row-wise and column-wise accesses of a warp are both conflict-free) and a [64][64] table
// tab[r][t] = W_4096^{r t}.
constexpr int F64_ROW = 65;
constexpr int F64_TILE = 64 * F64_ROW;            // float2 elements per transform

__device__ __forceinline__ void f64_bar(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }

// v[r] *= W^{S r t} (r = 1..63), then v[r] -> tile[r][t]  (end of a first pass)
template <int S> __device__ __forceinline__ void f64_twiddle_store(const float2 (&v)[64], float2* tile, const float2* tab, int t) {
  tile[t] = v[0];
#pragma unroll
  for (int r = 1; r < 64; ++r) tile[r * F64_ROW + t] = f64_cmul<(S > 0)>(v[r], tab[r * 64 + t]);
}
// v[c] <- tile[t][c]  (start of a second pass; in the order the first butterflies consume them: c = 8 a + b, b outermost)
__device__ __forceinline__ void f64_load_row(float2 (&v)[64], const float2* tile, int t) {
#pragma unroll
  for (int b = 0; b < 8; ++b)
#pragma unroll
    for (int a = 0; a < 8; ++a) v[8 * a + b] = tile[t * F64_ROW + 8 * a + b];
}
// tab[r][t] = W_4096^{r t} from the context's table tw[q] = exp(-2 pi i q / 8192)
__device__ __forceinline__ void f64_fill_tab(float2* tab, const float2* __restrict__ tw, int tid, int nthreads) {
  for (int i = tid; i < 4096; i += nthreads) tab[i] = tw[2 * (((i >> 6) * (i & 63)) & 4095)];
}
