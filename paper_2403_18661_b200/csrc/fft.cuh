// Shared-memory power-of-two complex FFT (Stockham autosort, radix 16/8/4/2 butterflies held in
// registers) used by the Welch, filter-design and overlap-save whitening kernels.
//
// Forward transform only, X[k] = sum_n x[n] exp(-2 pi i n k / M); callers get the inverse by
// conjugating input and output (IFFT(x) = conj(FFT(conj(x))) / M).
//
// Data lives in shared memory as T2 (float2 / double2) at padded positions fft_pad(i) = i + (i >> 4),
// which makes the stride-R scatter of each pass bank-conflict free for 8-byte elements.
// Twiddles come from a global table tw[q] = exp(-2 pi i q / AF_TW_N), computed on the host in double.
#pragma once

#include "common.cuh"

__host__ __device__ constexpr int fft_pad(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int fft_smem_elems(int m) { return m + (m >> 4) + 1; }

template <typename T2> struct scalar_of;
template <> struct scalar_of<float2> { using type = float; };
template <> struct scalar_of<double2> { using type = double; };

template <typename T2> __device__ __forceinline__ T2 mk2(typename scalar_of<T2>::type x, typename scalar_of<T2>::type y) {
  T2 r; r.x = x; r.y = y; return r;
}
template <typename T2> __device__ __forceinline__ T2 cadd(T2 a, T2 b) { return mk2<T2>(a.x + b.x, a.y + b.y); }
template <typename T2> __device__ __forceinline__ T2 csub(T2 a, T2 b) { return mk2<T2>(a.x - b.x, a.y - b.y); }
template <typename T2> __device__ __forceinline__ T2 cmul(T2 a, T2 b) {
  return mk2<T2>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename T2> __device__ __forceinline__ T2 cconj(T2 a) { return mk2<T2>(a.x, -a.y); }

// exp(-2 pi i idx / 16), idx = 0..7, as compile-time constants
template <typename T2> __device__ __forceinline__ T2 root16(int idx) {
  using T = typename scalar_of<T2>::type;
  const T c1 = (T)0.92387953251128673848, s1 = (T)0.38268343236508978178, h = (T)0.70710678118654752440;
  switch (idx) {
    case 0: return mk2<T2>((T)1, (T)0);
    case 1: return mk2<T2>(c1, -s1);
    case 2: return mk2<T2>(h, -h);
    case 3: return mk2<T2>(s1, -c1);
    case 4: return mk2<T2>((T)0, (T)-1);
    case 5: return mk2<T2>(-s1, -c1);
    case 6: return mk2<T2>(-h, -h);
    default: return mk2<T2>(-c1, -s1);
  }
}

// In-register forward DFT of R points, natural order in and out (recursive radix-2 DIT, fully unrolled).
template <int R, typename T2> struct RegFFT {
  static __device__ __forceinline__ void run(T2* v) {
    T2 e[R / 2], o[R / 2];
#pragma unroll
    for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
    RegFFT<R / 2, T2>::run(e);
    RegFFT<R / 2, T2>::run(o);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
      const int idx = k * (16 / R);
      T2 t;
      if (idx == 0) t = o[k];
      else if (idx == 4) t = mk2<T2>(o[k].y, -o[k].x);   // * (-i)
      else t = cmul(o[k], root16<T2>(idx));
      v[k] = cadd(e[k], t);
      v[k + R / 2] = csub(e[k], t);
    }
  }
};
template <typename T2> struct RegFFT<1, T2> {
  static __device__ __forceinline__ void run(T2*) {}
};

__host__ __device__ constexpr int fft_next_radix(int rem) {
  return (rem >= 256 || rem == 16) ? 16 : (rem == 128 ? 16 : (rem == 64 ? 8 : (rem == 32 ? 8 : rem)));
}

// One Stockham pass: length-NS sub-transforms -> length NS*R.
template <typename T2, int M, int R, int NS, int NT>
__device__ __forceinline__ void fft_pass(T2* s, const T2* __restrict__ tw, int tid) {
  constexpr int J = M / R;
  constexpr int JPT = (J + NT - 1) / NT;
  T2 v[JPT][R];
#pragma unroll
  for (int jj = 0; jj < JPT; ++jj) {
    const int j = tid + jj * NT;
    if (j < J) {
#pragma unroll
      for (int r = 0; r < R; ++r) v[jj][r] = s[fft_pad(j + r * J)];
      if (NS > 1) {
        // twiddles w^r, r = 1..R-1, w = exp(-2 pi i (j % NS) / (NS R)): ONE table load, the powers by a depth-4
        // product tree (w2 = w w, w4 = w2 w2, w8 = w4 w4, the rest as products of two of those): the table loads of all
        // R-1 powers made this pass wait on L1/L2 (long-scoreboard stalls); the tree costs R-2 complex multiplies and
        // loses < R ulp.
        const int q = (j % NS) * (AF_TW_N / (NS * R));
        T2 w[R];
        w[1] = tw[q];
        if (R > 2) w[2] = cmul(w[1], w[1]);
        if (R > 4) w[4] = cmul(w[2], w[2]);
        if (R > 8) w[8] = cmul(w[4], w[4]);
#pragma unroll
        for (int r = 3; r < R; ++r)
          if ((r & (r - 1)) != 0) {                 // not a power of two: highest set bit times the rest
            const int hb = r >= 8 ? 8 : (r >= 4 ? 4 : 2);
            w[r] = cmul(w[hb], w[r - hb]);
          }
#pragma unroll
        for (int r = 1; r < R; ++r) v[jj][r] = cmul(v[jj][r], w[r]);
      }
      RegFFT<R, T2>::run(v[jj]);
    }
  }
  __syncthreads();
#pragma unroll
  for (int jj = 0; jj < JPT; ++jj) {
    const int j = tid + jj * NT;
    if (j < J) {
      const int base = (j / NS) * (NS * R) + (j % NS);
#pragma unroll
      for (int r = 0; r < R; ++r) s[fft_pad(base + r * NS)] = v[jj][r];
    }
  }
  __syncthreads();
}

template <typename T2, int M, int NS, int NT> struct FftPasses {
  static __device__ __forceinline__ void run(T2* s, const T2* __restrict__ tw, int tid) {
    constexpr int R = fft_next_radix(M / NS);
    fft_pass<T2, M, R, NS, NT>(s, tw, tid);
    FftPasses<T2, M, NS * R, NT>::run(s, tw, tid);
  }
};
template <typename T2, int M, int NT> struct FftPasses<T2, M, M, NT> {
  static __device__ __forceinline__ void run(T2*, const T2* __restrict__, int) {}
};

// In-place forward FFT of the M complex values s[fft_pad(0..M-1)].  All NT threads of the block must
// call it; the caller must __syncthreads() after writing s and may read s right after it returns.
template <typename T2, int M, int NT>
__device__ __forceinline__ void fft_smem(T2* s, const T2* __restrict__ tw, int tid) {
  static_assert((M & (M - 1)) == 0 && M >= 16 && M <= AF_TW_N, "power of two, 16..8192");
  FftPasses<T2, M, 1, NT>::run(s, tw, tid);
}
