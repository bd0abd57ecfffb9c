// split_f32.cu -- fp32 operands for the tcgen05 GEMM by three-way bf16 splitting (SURVEY.md 8(f)
// NEXT #4: "a tcgen05 fp32 mode by 3-way bf16 operand splitting").
//
// A binary32 value x is the exact sum of three bf16 values (8 + 8 + 8 significand bits)
//     x0 = bf16(x),  x1 = bf16(x - x0),  x2 = bf16(x - x0 - x1)        (both differences are exact)
// so a product a.b = sum_{i,j} a_i b_j.  The six terms with i + j <= 2 carry everything above
// 2^-24 |a b|; the tensor core forms each exactly (8 x 8 bits) and adds in fp32.  The six partial
// GEMMs are ONE bf16 GEMM over a K six times as long: the operands are written K-concatenated,
//     A' = [A1 | A0 | A2 | A0 | A1 | A0],   B' = [B1 | B2 | B0 | B1 | B0 | B0]     (planes of A, B)
// smallest terms first, so that they meet an accumulator of their own magnitude.
#include "internal.h"

#include <algorithm>

namespace pinsage {
namespace {

__device__ __forceinline__ void split3(float x, __nv_bfloat16 &p0, __nv_bfloat16 &p1, __nv_bfloat16 &p2)
{
    p0 = __float2bfloat16_rn(x);
    const float r1 = x - __bfloat162float(p0);
    p1 = __float2bfloat16_rn(r1);
    const float r2 = r1 - __bfloat162float(p1);
    p2 = __float2bfloat16_rn(r2);
}

__device__ __forceinline__ uint2 pack4(const __nv_bfloat16 (&v)[4])
{
    __nv_bfloat162 lo = __halves2bfloat162(v[0], v[1]), hi = __halves2bfloat162(v[2], v[3]);
    return make_uint2(*reinterpret_cast<unsigned *>(&lo), *reinterpret_cast<unsigned *>(&hi));
}

// out[r, t*kt + c] = plane_{sel(t)}([S1 | S2][r, c]),  kt = K1 + K2, four columns per thread
template <bool IS_B>
__global__ void __launch_bounds__(256)
split3_kernel(const float *__restrict__ S1, int K1, long long ld1, const float *__restrict__ S2, int K2,
              long long ld2, long long rows, __nv_bfloat16 *__restrict__ out)
{
    const int kt = K1 + K2, groups = kt >> 2;
    const long long total = rows * groups;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long r = e / groups;
        const int c = (int)(e - r * groups) << 2;
        const float *src = c < K1 ? S1 + r * ld1 + c : S2 + r * ld2 + (c - K1);
        const float4 x = *reinterpret_cast<const float4 *>(src);
        __nv_bfloat16 p[3][4];
        split3(x.x, p[0][0], p[1][0], p[2][0]);
        split3(x.y, p[0][1], p[1][1], p[2][1]);
        split3(x.z, p[0][2], p[1][2], p[2][2]);
        split3(x.w, p[0][3], p[1][3], p[2][3]);
        const uint2 q0 = pack4(p[0]), q1 = pack4(p[1]), q2 = pack4(p[2]);
        uint2 *o = reinterpret_cast<uint2 *>(out + r * 6 * kt + c);
        const int step = kt >> 2;                                  // one term further, in uint2 units
        if (IS_B) {                                                // B' = [B1 | B2 | B0 | B1 | B0 | B0]
            o[0] = q1;
            o[step] = q2;
            o[2 * step] = q0;
            o[3 * step] = q1;
            o[4 * step] = q0;
            o[5 * step] = q0;
        } else {                                                   // A' = [A1 | A0 | A2 | A0 | A1 | A0]
            o[0] = q1;
            o[step] = q0;
            o[2 * step] = q2;
            o[3 * step] = q0;
            o[4 * step] = q1;
            o[5 * step] = q0;
        }
    }
}

}  // namespace

// S1 [rows x K1] (row stride ld1), S2 [rows x K2] (ld2) or null; K1, K2, ld1, ld2 multiples of 4,
// rows 16-byte aligned.  out: [rows x 6 (K1 + K2)] bf16.
cudaError_t launch_split3(bool is_b, const float *S1, int32_t K1, int64_t ld1, const float *S2, int32_t K2,
                          int64_t ld2, int64_t rows, void *out, cudaStream_t s, int *launches)
{
    if (rows <= 0) return cudaSuccess;
    const long long total = rows * ((K1 + K2) >> 2);
    const unsigned grid = (unsigned)std::max<long long>(1, std::min<long long>((total + 255) / 256, 148LL * 64));
    __nv_bfloat16 *o = static_cast<__nv_bfloat16 *>(out);
    if (is_b) split3_kernel<true><<<grid, 256, 0, s>>>(S1, K1, ld1, S2, K2, ld2, rows, o);
    else split3_kernel<false><<<grid, 256, 0, s>>>(S1, K1, ld1, S2, K2, ld2, rows, o);
    if (launches) ++*launches;
    return cudaGetLastError();
}

}  // namespace pinsage
