// gemm_simt.cu -- SIMT fp32-FMA GEMM with the path's epilogues.
//
// This is the PINSAGE_F32 mode (fp32 storage + IEEE fp32 FMA; tcgen05 kind::tf32 has a 10-bit
// mantissa and cannot meet the 1e-4 gate), and, for bf16 storage, the slow reference kernels
// selected by the context option "gemm_impl" = 1 (used to cross-check the tcgen05 kernels on
// all rows).  Computes S1/S3/S4/S5 of include/pinsage.h:
//   out = epi(A1 * B[:, :K1]^T + A2 * B[:, K1:]^T + bias)
// 64x64 tile, BK = 8, 256 threads, 4x4 micro-tile per thread.  When the row L2 norm is requested
// the un-normalised fp32 z goes to a scratch buffer and a second kernel (one warp per row)
// normalises and rounds once -- so out may alias A1 (the in-place layer).
#include "internal.h"

namespace pinsage {
namespace {

constexpr int BM = 64, BN = 64, BK = 8;

template <typename T>
__device__ __forceinline__ float2 load2(const T *p);
template <>
__device__ __forceinline__ float2 load2<float>(const float *p)
{
    return *reinterpret_cast<const float2 *>(p);
}
template <>
__device__ __forceinline__ float2 load2<__nv_bfloat16>(const __nv_bfloat16 *p)
{
    return __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162 *>(p));
}

template <typename T>
__device__ __forceinline__ float load1(const T *p);
template <>
__device__ __forceinline__ float load1<float>(const float *p)
{
    return *p;
}
template <>
__device__ __forceinline__ float load1<__nv_bfloat16>(const __nv_bfloat16 *p)
{
    return __bfloat162float(*p);
}

template <typename T>
__device__ __forceinline__ void store1(T *p, float v);
template <>
__device__ __forceinline__ void store1<float>(float *p, float v)
{
    *p = v;
}
template <>
__device__ __forceinline__ void store1<__nv_bfloat16>(__nv_bfloat16 *p, float v)
{
    *p = __float2bfloat16_rn(v);
}

// TOut = T (final) or float (scratch for the normalisation pass)
template <typename T, typename TOut>
__global__ void __launch_bounds__(256)
gemm_simt_kernel(const T *__restrict__ A1, const T *__restrict__ A2, const T *__restrict__ B,
                 const T *__restrict__ addend, const float *__restrict__ bias, TOut *__restrict__ out,
                 long long M, int K1, int K2, int N, int ldb, int relu, int Nb)
{
    __shared__ float As[BK][BM + 4];
    __shared__ float Bs[BK][BN + 4];
    const int tid = threadIdx.x;
    const int tx = tid % 16, ty = tid / 16;
    const long long row0 = (long long)blockIdx.x * BM;
    const int col0 = blockIdx.y * BN;
    const int Kt = K1 + K2;
    const int lr = tid / 4;        // 0..63: tile row (A) / tile col (B) this thread loads
    const int lk = (tid % 4) * 2;  // 0,2,4,6
    float acc[4][4] = {};
    for (int k0 = 0; k0 < Kt; k0 += BK) {
        // K1 and K2 are multiples of 8 = BK, so a K tile never straddles the two segments
        const bool seg2 = k0 >= K1;
        const T *A = seg2 ? A2 : A1;
        const int lda = seg2 ? K2 : K1;
        const int ka = seg2 ? k0 - K1 : k0;
        float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
        if (row0 + lr < M) a = load2<T>(A + (size_t)(row0 + lr) * lda + ka + lk);
        if (col0 + lr < Nb) b = load2<T>(B + (size_t)(col0 + lr) * ldb + k0 + lk);   // Nb = rows of B that exist
        As[lk][lr] = a.x;
        As[lk + 1][lr] = a.y;
        Bs[lk][lr] = b.x;
        Bs[lk + 1][lr] = b.y;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < BK; ++k) {
            float av[4], bv[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) av[i] = As[k][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) bv[j] = Bs[k][tx * 4 + j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long long r = row0 + ty * 4 + i;
        if (r >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = col0 + tx * 4 + j;
            if (c >= N) continue;
            float v = acc[i][j];
            if (addend) v += load1<T>(addend + (size_t)r * N + c);
            if (bias) v += bias[c];
            if (relu) v = fmaxf(v, 0.f);
            store1<TOut>(out + (size_t)r * N + c, v);
        }
    }
}

// One warp per row: out = z / ||z||_2 (zero row stays zero), rounded once to T.
template <typename T>
__global__ void __launch_bounds__(256)
rownorm_kernel(const float *__restrict__ z, T *__restrict__ out, long long M, int N)
{
    const long long row = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= M) return;
    const int lane = threadIdx.x & 31;
    const float *zr = z + (size_t)row * N;
    float ss = 0.f;
    for (int c = lane; c < N; c += 32) ss = fmaf(zr[c], zr[c], ss);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    const float inv = ss > 0.f ? 1.0f / sqrtf(ss) : 0.f;
    for (int c = lane; c < N; c += 32) store1<T>(out + (size_t)row * N + c, zr[c] * inv);
}

template <typename T>
cudaError_t run(const GemmArgs &a, float *ztmp, cudaStream_t s, int *launches)
{
    const long long mb = (a.M + BM - 1) / BM;
    if (mb > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)mb, (unsigned)((a.N + BN - 1) / BN));
    const T *A1 = static_cast<const T *>(a.A1), *A2 = static_cast<const T *>(a.A2);
    const T *B = static_cast<const T *>(a.B);
    const T *add = static_cast<const T *>(a.addend);
    const int ldb = a.ldb > 0 ? a.ldb : a.K1 + a.K2;
    const int Nb = a.b_rows > 0 ? (int)a.b_rows : a.N;
    if (a.l2norm) {
        if (!ztmp) return cudaErrorInvalidValue;
        gemm_simt_kernel<T, float><<<grid, 256, 0, s>>>(A1, A2, B, add, a.bias, ztmp, a.M, a.K1, a.K2,
                                                        a.N, ldb, a.relu, Nb);
        const long long rb = (a.M + 7) / 8;
        rownorm_kernel<T><<<(unsigned)rb, 256, 0, s>>>(ztmp, static_cast<T *>(a.out), a.M, a.N);
        if (launches) *launches += 2;
    } else if (a.out_f32) {
        gemm_simt_kernel<T, float><<<grid, 256, 0, s>>>(A1, A2, B, add, a.bias, static_cast<float *>(a.out),
                                                        a.M, a.K1, a.K2, a.N, ldb, a.relu, Nb);
        if (launches) *launches += 1;
    } else {
        gemm_simt_kernel<T, T><<<grid, 256, 0, s>>>(A1, A2, B, add, a.bias, static_cast<T *>(a.out),
                                                    a.M, a.K1, a.K2, a.N, ldb, a.relu, Nb);
        if (launches) *launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace

size_t gemm_simt_scratch_bytes(const GemmArgs &a)
{
    return a.l2norm ? (size_t)a.M * (size_t)a.N * sizeof(float) : 0;
}

cudaError_t launch_gemm_simt(DType dt, const GemmArgs &a, float *ztmp, cudaStream_t s, int *launches)
{
    if (a.M <= 0) return cudaSuccess;
    return dt == DType::BF16 ? run<__nv_bfloat16>(a, ztmp, s, launches)
                             : run<float>(a, ztmp, s, launches);
}

}  // namespace pinsage
