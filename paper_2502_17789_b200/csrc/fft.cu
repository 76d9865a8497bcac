// Subgrid FFT: steps a4 / a7.  Centred L x L DFT of one plane per block, in shared memory,
// scaled by 1/L^2 (Eq. 7-8 :107-117, :157, :170; R1, R2).
//
// For L a multiple of 4 the centred transform equals checkerboard * FFT * checkerboard
// ((-1)^(x+y) on input and output), so the kernel is a plain in-place mixed-radix
// decimation-in-time FFT: the load from global memory applies the checkerboard and the
// digit-reversal permutation of both axes, the row and column passes then run in place with
// radix-4/2/3 butterflies, and the store applies the checkerboard and the 1/L^2.
#include "kernels.h"

namespace idg {

namespace {

// radix of stage s (stage 0 first, sub-transform size 1) for each supported L
template <int L>
__host__ __device__ constexpr int radix(int s) {
  return L == 32   ? (s < 2 ? 4 : (s == 2 ? 2 : 1))
         : L == 64 ? (s < 3 ? 4 : 1)
         : L == 96 ? (s < 2 ? 4 : (s == 2 ? 2 : (s == 3 ? 3 : 1)))
                   : (s < 3 ? 4 : (s == 3 ? 2 : 1));
}
template <int L>
__host__ __device__ constexpr int n_stages() { return (L == 32 || L == 64) ? 3 : 4; }

// position of natural index n in the digit-reversed input order of the in-place DIT:
// pos_N(n) = (n mod r_k) * N_{k-1} + pos_{N_{k-1}}(n div r_k), r_k the radix of the last stage.
template <int L>
__host__ __device__ constexpr int dit_position(int n) {
  int pos = 0;
  int size = L;
  for (int s = n_stages<L>() - 1; s >= 0; --s) {
    const int r = radix<L>(s);
    size /= r;
    pos += (n % r) * size;
    n /= r;
  }
  return pos;
}

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// One radix-R DIT stage over `lines` independent length-L lines.  Element e of line q lives at
// data[q * line_stride + e * elem_stride].  m = product of the radices already done.
// tw[k] = exp(-+ 2 pi i k / L).  SIGN = -1 forward, +1 inverse.
template <int L, int R, int M, int SIGN, int T>
__device__ __forceinline__ void fft_stage(float2* data, const float2* tw, int line_stride, int elem_stride) {
  constexpr int m = M;
  constexpr int BF = L / R;              // butterflies per line
  const int total = BF * L;              // L lines
  for (int idx = threadIdx.x; idx < total; idx += T) {
    const int line = idx % L, bf = idx / L;   // consecutive threads take consecutive lines
    const int j = bf % m;
    const int blk = bf / m;
    float2* p = data + line * line_stride + (blk * m * R + j) * elem_stride;
    const int tstep = j * (L / (m * R));   // twiddle index step: w_{mR}^{j q} = tw[j q L/(mR)]
    float2 x[R];
#pragma unroll
    for (int q = 0; q < R; ++q) {
      x[q] = p[q * m * elem_stride];
      if (q > 0) x[q] = cmulf(x[q], tw[q * tstep]);
    }
    if (R == 2) {
      const float2 a = x[0], b = x[1];
      x[0] = make_float2(a.x + b.x, a.y + b.y);
      x[1] = make_float2(a.x - b.x, a.y - b.y);
    } else if (R == 4) {
      const float2 s02 = make_float2(x[0].x + x[2].x, x[0].y + x[2].y);
      const float2 d02 = make_float2(x[0].x - x[2].x, x[0].y - x[2].y);
      const float2 s13 = make_float2(x[1].x + x[3].x, x[1].y + x[3].y);
      const float2 d13 = make_float2(x[1].x - x[3].x, x[1].y - x[3].y);
      // SIGN*i * d13 : forward (-i): (d.y, -d.x); inverse (+i): (-d.y, d.x)
      const float2 r13 = SIGN < 0 ? make_float2(d13.y, -d13.x) : make_float2(-d13.y, d13.x);
      x[0] = make_float2(s02.x + s13.x, s02.y + s13.y);
      x[1] = make_float2(d02.x + r13.x, d02.y + r13.y);
      x[2] = make_float2(s02.x - s13.x, s02.y - s13.y);
      x[3] = make_float2(d02.x - r13.x, d02.y - r13.y);
    } else if (R == 3) {
      // y0 = x0+x1+x2; y1 = x0 + w x1 + w^2 x2; y2 = x0 + w^2 x1 + w x2, w = exp(SIGN 2 pi i/3)
      const float hs = SIGN * 0.86602540378443864676f;   // Im(w)
      const float2 s = make_float2(x[1].x + x[2].x, x[1].y + x[2].y);
      const float2 d = make_float2(x[1].x - x[2].x, x[1].y - x[2].y);
      const float2 c = make_float2(fmaf(-0.5f, s.x, x[0].x), fmaf(-0.5f, s.y, x[0].y));
      // i*hs*d = (-hs d.y, hs d.x)
      const float2 e = make_float2(-hs * d.y, hs * d.x);
      x[0] = make_float2(x[0].x + s.x, x[0].y + s.y);
      x[1] = make_float2(c.x + e.x, c.y + e.y);
      x[2] = make_float2(c.x - e.x, c.y - e.y);
    }
#pragma unroll
    for (int q = 0; q < R; ++q) p[q * m * elem_stride] = x[q];
  }
}

template <int L, int SIGN, int T, int S, int M>
struct Pass {
  static __device__ __forceinline__ void run(float2* data, const float2* tw, int line_stride, int elem_stride) {
    constexpr int R = radix<L>(S);
    fft_stage<L, R, M, SIGN, T>(data, tw, line_stride, elem_stride);
    __syncthreads();
    Pass<L, SIGN, T, S + 1, M * R>::run(data, tw, line_stride, elem_stride);
  }
};
template <int L, int SIGN, int T, int S>
struct Pass<L, SIGN, T, S, L> {
  static __device__ __forceinline__ void run(float2*, const float2*, int, int) {}
};

template <int L, int SIGN, int T>
__global__ void __launch_bounds__(T) fft_kernel(float2* __restrict__ planes) {
  constexpr int PITCH = L + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* data = reinterpret_cast<float2*>(smem_raw);          // [L][PITCH]
  float2* tw = data + L * PITCH;                               // [L]
  int* pos = reinterpret_cast<int*>(tw + L);                   // [L]
  float2* plane = planes + static_cast<int64_t>(blockIdx.x) * L * L;

  for (int k = threadIdx.x; k < L; k += T) {
    float s, c;
    sincospif(2.0f * k / L, &s, &c);
    tw[k] = make_float2(c, SIGN * s);
    pos[k] = dit_position<L>(k);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < L * L; i += T) {
    const int y = i / L, x = i % L;
    float2 v = plane[i];
    if ((x + y) & 1) v = make_float2(-v.x, -v.y);
    data[pos[y] * PITCH + pos[x]] = v;
  }
  __syncthreads();
  // rows: element stride 1, lines = rows; consecutive threads take consecutive rows
  Pass<L, SIGN, T, 0, 1>::run(data, tw, PITCH, 1);
  // columns: element stride PITCH, lines = columns; consecutive threads take consecutive columns
  Pass<L, SIGN, T, 0, 1>::run(data, tw, 1, PITCH);
  const float scale = 1.0f / (L * L);
  for (int i = threadIdx.x; i < L * L; i += T) {
    const int y = i / L, x = i % L;
    float2 v = data[y * PITCH + x];
    const float sc = ((x + y) & 1) ? -scale : scale;
    plane[i] = make_float2(v.x * sc, v.y * sc);
  }
}

template <int L>
cudaError_t launch(int64_t n_planes, float2* planes, int direction, cudaStream_t stream) {
  constexpr int T = 256;
  const size_t smem = static_cast<size_t>(L) * (L + 1) * sizeof(float2) + L * sizeof(float2) + L * sizeof(int);
  if (n_planes == 0) return cudaSuccess;
  cudaError_t e;
  if (direction > 0) {
    e = cudaFuncSetAttribute(fft_kernel<L, -1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    fft_kernel<L, -1, T><<<static_cast<unsigned>(n_planes), T, smem, stream>>>(planes);
  } else {
    e = cudaFuncSetAttribute(fft_kernel<L, +1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    fft_kernel<L, +1, T><<<static_cast<unsigned>(n_planes), T, smem, stream>>>(planes);
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_subgrid_fft(int L, int64_t n_planes, float2* planes, int direction, cudaStream_t stream) {
  switch (L) {
    case 32:  return launch<32>(n_planes, planes, direction, stream);
    case 64:  return launch<64>(n_planes, planes, direction, stream);
    case 96:  return launch<96>(n_planes, planes, direction, stream);
    case 128: return launch<128>(n_planes, planes, direction, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
