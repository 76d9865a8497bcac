// Subgrid FFT: steps a4 / a7.  Centred L x L DFT of one plane per block, scaled by 1/L^2
// (Eq. 7-8 :107-117, :157, :170; R1, R2).
//
// For even L the centred transform equals checkerboard * DFT * checkerboard ((-1)^(x+y) on input and
// output), so the kernel is a plain 2-D FFT with the checkerboard folded into the global load and
// the checkerboard and 1/L^2 into the global store.
//
// Every 1-D transform of length L = 8 R2 (R2 = 4, 6, 8, 12, 16, 20: L = 32, 48, 64, 96, 128, 160, the range of
// PAPER.md Fig. 7 :363-369) is two register-resident steps:
//   n = n1 R2 + n2, k = k1 + 8 k2:
//   step 1  Y[k1][n2] = w_L^(n2 k1) * sum_n1 x[n1 R2 + n2] w_8^(n1 k1)     (radix-8 butterfly per n2)
//   step 2  X[k1 + 8 k2] = sum_n2 Y[k1][n2] w_R2^(n2 k2)                   (radix-R2 butterfly per k1)
// A plane therefore makes one trip global -> registers (row step 1) -> shared -> registers (row step
// 2) -> shared -> registers (column step 1, in place) -> shared -> registers (column step 2) -> global:
// three shared-memory round trips and three block barriers, against one round trip per radix-4 stage
// before.  Row step 2 is the only step whose tasks read and write different positions of a line; a
// warp owns whole rows there, so a warp-level barrier between its reads and writes is enough.
#include "kernels.h"

namespace idg {

namespace {

__device__ __forceinline__ float2 cadd2(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub2(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// multiply by SIGN * i  (forward: -i)
template <int SIGN>
__device__ __forceinline__ float2 rot90(float2 d) {
  return SIGN < 0 ? make_float2(d.y, -d.x) : make_float2(-d.y, d.x);
}
// exp(SIGN 2 pi i m / N) for the small transforms; the tables fold to immediates once unrolled
template <int N, int SIGN>
__device__ __forceinline__ float2 wsmall(int m) {
  if constexpr (N == 8) {
    const float c[8] = {1.f, 0.707106781f, 0.f, -0.707106781f, -1.f, -0.707106781f, 0.f, 0.707106781f};
    const float s[8] = {0.f, 0.707106781f, 1.f, 0.707106781f, 0.f, -0.707106781f, -1.f, -0.707106781f};
    return make_float2(c[m], SIGN * s[m]);
  } else if constexpr (N == 6) {
    const float c[6] = {1.f, 0.5f, -0.5f, -1.f, -0.5f, 0.5f};
    const float s[6] = {0.f, 0.866025404f, 0.866025404f, 0.f, -0.866025404f, -0.866025404f};
    return make_float2(c[m], SIGN * s[m]);
  } else if constexpr (N == 20) {
    const float c[20] = {1.f, 0.951056516f, 0.809016994f, 0.587785252f, 0.309016994f, 0.f, -0.309016994f,
                         -0.587785252f, -0.809016994f, -0.951056516f, -1.f, -0.951056516f, -0.809016994f,
                         -0.587785252f, -0.309016994f, 0.f, 0.309016994f, 0.587785252f, 0.809016994f, 0.951056516f};
    const float s[20] = {0.f, 0.309016994f, 0.587785252f, 0.809016994f, 0.951056516f, 1.f, 0.951056516f,
                         0.809016994f, 0.587785252f, 0.309016994f, 0.f, -0.309016994f, -0.587785252f,
                         -0.809016994f, -0.951056516f, -1.f, -0.951056516f, -0.809016994f, -0.587785252f,
                         -0.309016994f};
    return make_float2(c[m], SIGN * s[m]);
  } else if constexpr (N == 12) {
    const float c[12] = {1.f, 0.866025404f, 0.5f, 0.f, -0.5f, -0.866025404f, -1.f, -0.866025404f, -0.5f, 0.f, 0.5f,
                         0.866025404f};
    const float s[12] = {0.f, 0.5f, 0.866025404f, 1.f, 0.866025404f, 0.5f, 0.f, -0.5f, -0.866025404f, -1.f,
                         -0.866025404f, -0.5f};
    return make_float2(c[m], SIGN * s[m]);
  } else {
    const float c[16] = {1.f, 0.923879533f, 0.707106781f, 0.382683432f, 0.f, -0.382683432f, -0.707106781f,
                         -0.923879533f, -1.f, -0.923879533f, -0.707106781f, -0.382683432f, 0.f, 0.382683432f,
                         0.707106781f, 0.923879533f};
    const float s[16] = {0.f, 0.382683432f, 0.707106781f, 0.923879533f, 1.f, 0.923879533f, 0.707106781f,
                         0.382683432f, 0.f, -0.382683432f, -0.707106781f, -0.923879533f, -1.f, -0.923879533f,
                         -0.707106781f, -0.382683432f};
    return make_float2(c[m], SIGN * s[m]);
  }
}

// ---- small DFTs on registers, natural order in and out: X[k] = sum_n x[n] exp(SIGN 2 pi i n k / N)
template <int SIGN>
__device__ __forceinline__ void dft2(float2& a, float2& b) {
  const float2 s = cadd2(a, b), d = csub2(a, b);
  a = s; b = d;
}
template <int SIGN>
__device__ __forceinline__ void dft3(float2& x0, float2& x1, float2& x2) {
  const float hs = SIGN * 0.86602540378443864676f;   // Im exp(SIGN 2 pi i / 3)
  const float2 s = cadd2(x1, x2), d = csub2(x1, x2);
  const float2 c = make_float2(fmaf(-0.5f, s.x, x0.x), fmaf(-0.5f, s.y, x0.y));
  const float2 e = make_float2(-hs * d.y, hs * d.x);  // i hs d
  x0 = cadd2(x0, s); x1 = cadd2(c, e); x2 = csub2(c, e);
}
template <int SIGN>
__device__ __forceinline__ void dft4(float2& x0, float2& x1, float2& x2, float2& x3) {
  const float2 a = cadd2(x0, x2), b = csub2(x0, x2), c = cadd2(x1, x3), d = rot90<SIGN>(csub2(x1, x3));
  x0 = cadd2(a, c); x1 = cadd2(b, d); x2 = csub2(a, c); x3 = csub2(b, d);
}
// X[k] = sum x[n] w^(nk), w = exp(SIGN 2 pi i / 5): conjugate pairs (1, 4) and (2, 3)
template <int SIGN>
__device__ __forceinline__ void dft5(float2& x0, float2& x1, float2& x2, float2& x3, float2& x4) {
  const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;          // cos 2 pi/5, cos 4 pi/5
  const float s1 = SIGN * 0.95105651629515357212f, s2 = SIGN * 0.58778525229247312917f;   // sin 2 pi/5, sin 4 pi/5
  const float2 p1 = cadd2(x1, x4), d1 = csub2(x1, x4), p2 = cadd2(x2, x3), d2 = csub2(x2, x3);
  const float2 a1 = make_float2(fmaf(c1, p1.x, fmaf(c2, p2.x, x0.x)), fmaf(c1, p1.y, fmaf(c2, p2.y, x0.y)));
  const float2 a2 = make_float2(fmaf(c2, p1.x, fmaf(c1, p2.x, x0.x)), fmaf(c2, p1.y, fmaf(c1, p2.y, x0.y)));
  const float2 e1 = make_float2(fmaf(s1, d1.x, s2 * d2.x), fmaf(s1, d1.y, s2 * d2.y));   // then times i
  const float2 e2 = make_float2(fmaf(s2, d1.x, -s1 * d2.x), fmaf(s2, d1.y, -s1 * d2.y));
  const float2 b1 = make_float2(-e1.y, e1.x), b2 = make_float2(-e2.y, e2.x);
  x0 = cadd2(x0, cadd2(p1, p2));
  x1 = cadd2(a1, b1); x4 = csub2(a1, b1);
  x2 = cadd2(a2, b2); x3 = csub2(a2, b2);
}
// N = P Q by the same index split as above: n = n1 Q + n2, k = k1 + P k2
template <int N, int SIGN>
__device__ __forceinline__ void dft_small(float2 (&x)[N]) {
  if constexpr (N == 4) {
    dft4<SIGN>(x[0], x[1], x[2], x[3]);
  } else if constexpr (N == 6) {                     // 6 = 2 x 3
    float2 y[6];                                     // y[k1 * 3 + n2]
#pragma unroll
    for (int n2 = 0; n2 < 3; ++n2) {
      float2 a = x[n2], b = x[3 + n2];
      dft2<SIGN>(a, b);
      y[n2] = a;
      y[3 + n2] = n2 ? cmulf(b, wsmall<6, SIGN>(n2)) : b;
    }
#pragma unroll
    for (int k1 = 0; k1 < 2; ++k1) {
      dft3<SIGN>(y[k1 * 3], y[k1 * 3 + 1], y[k1 * 3 + 2]);
#pragma unroll
      for (int k2 = 0; k2 < 3; ++k2) x[k1 + 2 * k2] = y[k1 * 3 + k2];
    }
  } else {
    constexpr int P = 4, Q = N / 4;                  // 8 = 4 x 2, 12 = 4 x 3, 16 = 4 x 4, 20 = 4 x 5
    float2 y[N];                                     // y[k1 * Q + n2]
#pragma unroll
    for (int n2 = 0; n2 < Q; ++n2) {
      float2 a = x[n2], b = x[Q + n2], c = x[2 * Q + n2], d = x[3 * Q + n2];
      dft4<SIGN>(a, b, c, d);
      y[n2] = a;
      y[Q + n2] = n2 ? cmulf(b, wsmall<N, SIGN>(n2)) : b;
      y[2 * Q + n2] = n2 ? cmulf(c, wsmall<N, SIGN>(2 * n2)) : c;
      y[3 * Q + n2] = n2 ? cmulf(d, wsmall<N, SIGN>(3 * n2)) : d;
    }
#pragma unroll
    for (int k1 = 0; k1 < P; ++k1) {
      if constexpr (Q == 2) {
        dft2<SIGN>(y[k1 * Q], y[k1 * Q + 1]);
      } else if constexpr (Q == 3) {
        dft3<SIGN>(y[k1 * Q], y[k1 * Q + 1], y[k1 * Q + 2]);
      } else if constexpr (Q == 5) {
        dft5<SIGN>(y[k1 * Q], y[k1 * Q + 1], y[k1 * Q + 2], y[k1 * Q + 3], y[k1 * Q + 4]);
      } else {
        dft4<SIGN>(y[k1 * Q], y[k1 * Q + 1], y[k1 * Q + 2], y[k1 * Q + 3]);
      }
#pragma unroll
      for (int k2 = 0; k2 < Q; ++k2) x[k1 + P * k2] = y[k1 * Q + k2];
    }
  }
}

template <int L>
struct FftThreads {
  static constexpr int value = L == 32 ? 128 : (L == 48 ? 192 : (L == 64 ? 256 : (L == 96 ? 576 : (L == 128 ? 512 : 640))));
};

// Where the transform reads its input: the plane itself (in place), or, for the prediction direction, the
// master grid patch under the subgrid (step a6, the splitter, fused into the load of step a7).
struct GridSource {
  const float2* grid;      // [W, 4, Ng, Ng]; nullptr = in place
  const int32_t* meta;     // subgrid metadata of plane 0's subgrid onwards
  int Ng;
};

template <int L, int SIGN>
__global__ void __launch_bounds__(FftThreads<L>::value) fft_kernel(float2* __restrict__ planes, const GridSource src) {
  constexpr int T = FftThreads<L>::value;
  constexpr int R2 = L / 8;
  // Row step 1 stores 8 groups of R2 + 1.  With the pitch = 8 (mod 16) float2, the 4 rows a warp touches in
  // the row steps land on complementary halves of the 16 8-byte bank slots: every access is conflict-free.
  constexpr int PITCH = L + 8;
  static_assert(R2 == 4 || R2 == 6 || R2 == 8 || R2 == 12 || R2 == 16 || R2 == 20, "L = 8 R2, R2 even");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* data = reinterpret_cast<float2*>(smem_raw);          // [L][PITCH]
  float2* tw = data + L * PITCH;                               // [L] exp(SIGN 2 pi i m / L)
  float2* plane = planes + static_cast<int64_t>(blockIdx.x) * L * L;
  const int tid = threadIdx.x;
  // input rows: `in` + r * in_pitch
  const float2* in = plane;
  int64_t in_pitch = L;
  if (src.grid != nullptr) {
    const int32_t* m = src.meta + static_cast<int64_t>(blockIdx.x >> 2) * kMetaStride;
    const int x0 = m[5], y0 = m[6], layer = m[11], pol = blockIdx.x & 3;
    in = src.grid + ((static_cast<int64_t>(layer) * 4 + pol) * src.Ng + y0) * src.Ng + x0;
    in_pitch = src.Ng;
  }

  for (int k = tid; k < L; k += T) {
    float s, c;
    sincospif(2.0f * k / L, &s, &c);
    tw[k] = make_float2(c, SIGN * s);
  }

  // ---- rows, step 1: global -> radix-8 over n1 -> twiddle -> shared [r][k1 (R2 + 1) + n2]
  // (the twiddle table is read only after the barrier below, so step 1 is split around it)
  constexpr int IT_R1 = (L * R2 + T - 1) / T;
  float2 xr[IT_R1][8];
#pragma unroll
  for (int it = 0; it < IT_R1; ++it) {
    const int t = tid + it * T, r = t / R2, n2 = t % R2;
    if (t < L * R2) {
      const float sg = ((r + n2) & 1) ? -1.f : 1.f;   // checkerboard; R2 is even, so n1 R2 drops out
#pragma unroll
      for (int n1 = 0; n1 < 8; ++n1) {
        const float2 v = in[r * in_pitch + n1 * R2 + n2];
        xr[it][n1] = make_float2(v.x * sg, v.y * sg);
      }
      dft_small<8, SIGN>(xr[it]);
    }
  }
  __syncthreads();                                    // twiddles ready
#pragma unroll
  for (int it = 0; it < IT_R1; ++it) {
    const int t = tid + it * T, r = t / R2, n2 = t % R2;
    if (t < L * R2) {
      float2* row = data + r * PITCH + n2;
      row[0] = xr[it][0];
#pragma unroll
      for (int k1 = 1; k1 < 8; ++k1) row[k1 * (R2 + 1)] = cmulf(xr[it][k1], tw[n2 * k1]);
    }
  }
  __syncthreads();

  // ---- rows, step 2: a warp owns 4 whole rows; read, warp barrier, radix-R2 over n2, write natural order
  constexpr int IT_R2 = (L * 8 + T - 1) / T;
#pragma unroll
  for (int it = 0; it < IT_R2; ++it) {
    const int t = tid + it * T, r = t >> 3, k1 = t & 7;
    if (t < L * 8) {                                  // warp-uniform: T and 8 L are multiples of 32
      float2 y[R2];
      const float2* src = data + r * PITCH + k1 * (R2 + 1);
#pragma unroll
      for (int n2 = 0; n2 < R2; ++n2) y[n2] = src[n2];
      __syncwarp();
      dft_small<R2, SIGN>(y);
      float2* dst = data + r * PITCH + k1;
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) dst[8 * k2] = y[k2];
    }
  }
  __syncthreads();

  // ---- columns, step 1 (in place): radix-8 over n1, twiddle; consecutive threads = consecutive columns
  constexpr int IT_C1 = (L * R2 + T - 1) / T;
#pragma unroll
  for (int it = 0; it < IT_C1; ++it) {
    const int t = tid + it * T, n2 = t / L, c = t % L;
    if (t < L * R2) {
      float2 x[8];
      float2* col = data + n2 * PITCH + c;
#pragma unroll
      for (int n1 = 0; n1 < 8; ++n1) x[n1] = col[n1 * R2 * PITCH];
      dft_small<8, SIGN>(x);
      col[0] = x[0];
#pragma unroll
      for (int k1 = 1; k1 < 8; ++k1) col[k1 * R2 * PITCH] = cmulf(x[k1], tw[n2 * k1]);
    }
  }
  __syncthreads();

  // ---- columns, step 2: radix-R2 over n2 -> checkerboard, 1/L^2 -> global (rows of 8 L bytes, coalesced)
  constexpr int IT_C2 = (L * 8 + T - 1) / T;
  const float scale = 1.0f / (L * L);
#pragma unroll
  for (int it = 0; it < IT_C2; ++it) {
    const int t = tid + it * T, k1 = t / L, c = t % L;
    if (t < L * 8) {
      float2 y[R2];
      const float2* col = data + k1 * R2 * PITCH + c;
#pragma unroll
      for (int n2 = 0; n2 < R2; ++n2) y[n2] = col[n2 * PITCH];
      dft_small<R2, SIGN>(y);
      const float sc = ((k1 + c) & 1) ? -scale : scale;   // 8 k2 is even
#pragma unroll
      for (int k2 = 0; k2 < R2; ++k2) plane[(k1 + 8 * k2) * L + c] = make_float2(y[k2].x * sc, y[k2].y * sc);
    }
  }
}

template <int L>
cudaError_t launch(int64_t n_planes, float2* planes, int direction, const GridSource& src, cudaStream_t stream) {
  constexpr int T = FftThreads<L>::value;
  const size_t smem = static_cast<size_t>(L) * (L + 8) * sizeof(float2) + L * sizeof(float2);
  if (n_planes == 0) return cudaSuccess;
  cudaError_t e;
  if (direction > 0) {
    e = cudaFuncSetAttribute(fft_kernel<L, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    fft_kernel<L, -1><<<static_cast<unsigned>(n_planes), T, smem, stream>>>(planes, src);
  } else {
    e = cudaFuncSetAttribute(fft_kernel<L, +1>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    fft_kernel<L, +1><<<static_cast<unsigned>(n_planes), T, smem, stream>>>(planes, src);
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_subgrid_fft(int L, int64_t n_planes, float2* planes, int direction, cudaStream_t stream) {
  const GridSource none{nullptr, nullptr, 0};
  switch (L) {
    case 32:  return launch<32>(n_planes, planes, direction, none, stream);
    case 48:  return launch<48>(n_planes, planes, direction, none, stream);
    case 64:  return launch<64>(n_planes, planes, direction, none, stream);
    case 96:  return launch<96>(n_planes, planes, direction, none, stream);
    case 128: return launch<128>(n_planes, planes, direction, none, stream);
    case 160: return launch<160>(n_planes, planes, direction, none, stream);
    default:  return cudaErrorInvalidValue;
  }
}

cudaError_t launch_split_ifft(const int32_t* meta, int64_t first, int64_t count, int L, int Ng, const float2* grid,
                              float2* subgrids, cudaStream_t stream) {
  const GridSource src{grid, meta + first * kMetaStride, Ng};
  switch (L) {
    case 32:  return launch<32>(count * 4, subgrids, -1, src, stream);
    case 48:  return launch<48>(count * 4, subgrids, -1, src, stream);
    case 64:  return launch<64>(count * 4, subgrids, -1, src, stream);
    case 96:  return launch<96>(count * 4, subgrids, -1, src, stream);
    case 128: return launch<128>(count * 4, subgrids, -1, src, stream);
    case 160: return launch<160>(count * 4, subgrids, -1, src, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
