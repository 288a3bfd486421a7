// The voxel update of Eq. 7 on a float4 column with packed fp32x2 arithmetic, shared by every
// fused kernel (idg_tma.cu, idg_stream.cu, idg_resident.cu).  Device code only; internal to libidg_b200.so.
#pragma once
#include "idg_kernels.cuh"
#include "idg_ptx.cuh"

namespace idg {

struct F4 { float x, y, z, w; };

__device__ __forceinline__ F4 lds4(const float *p)
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    return F4{v.x, v.y, v.z, v.w};
}
__device__ __forceinline__ void sts4(float *p, const F4 &a)
{
    *reinterpret_cast<float4 *>(p) = make_float4(a.x, a.y, a.z, a.w);
}

// Four voxel updates (Eq. 7) of one float4 column with packed fp32x2 arithmetic (FFMA2 / FADD2 /
// FMUL2: two IEEE fp32 results per issued instruction; each component rounds exactly like the
// scalar update() of idg_kernels.cuh, so results are bit-identical to the scalar kernels).
struct Consts {
    float2 w, ax, ay, az, s, one;
};
// s: 1/(K rms) for the intensity-driven conductance (Eq. 6); s^2/4 for the gradient-driven one (Eq. 5)
__device__ __forceinline__ Consts make_consts(float ax, float ay, float az, float s, float w)
{
    Consts k;
    k.w = make_float2(w, w);
    k.ax = make_float2(ax, ax);
    k.ay = make_float2(ay, ay);
    k.az = make_float2(az, az);
    k.s = make_float2(s, s);
    k.one = make_float2(1.0f, 1.0f);
    return k;
}
template <bool PM = false>
__device__ __forceinline__ Consts make_consts(const CubeParams &p)
{
    return make_consts(p.ax, p.ay, p.az, PM ? 0.25f * p.s * p.s : p.s, p.w);
}
__device__ __forceinline__ float2 update2(float2 c, float2 sx, float2 ym, float2 yp, float2 zm, float2 zp,
                                          const Consts &k)
{
    const float2 lap = __ffma2_rn(k.ax, sx, __ffma2_rn(k.ay, __fadd2_rn(yp, ym),
                                                        __ffma2_rn(k.az, __fadd2_rn(zp, zm), __fmul2_rn(k.w, c))));
    const float2 u = __fmul2_rn(c, k.s);
    const float2 den = __ffma2_rn(u, u, k.one);
    const float2 r = make_float2(ptx::rcp_approx(den.x), ptx::rcp_approx(den.y));
    return __ffma2_rn(lap, r, c);
}
// Gradient-driven variant (Eq. 5; readings P1-P3): conductance 1/(1 + q G), G = sum_j
// (I_{+j} - I_{-j})^2, q = s^2/4 (kept in k.s); same operation order as update_pm() of idg_kernels.cuh.
// gx = difference of the x neighbours.
__device__ __forceinline__ float2 update2_pm(float2 c, float2 sx, float2 gx, float2 ym, float2 yp, float2 zm,
                                             float2 zp, const Consts &k)
{
    const float2 neg = make_float2(-1.0f, -1.0f);
    const float2 lap = __ffma2_rn(k.ax, sx, __ffma2_rn(k.ay, __fadd2_rn(yp, ym),
                                                        __ffma2_rn(k.az, __fadd2_rn(zp, zm), __fmul2_rn(k.w, c))));
    const float2 gy = __ffma2_rn(neg, ym, yp), gz = __ffma2_rn(neg, zm, zp);
    const float2 G = __ffma2_rn(gz, gz, __ffma2_rn(gy, gy, __fmul2_rn(gx, gx)));
    const float2 den = __ffma2_rn(k.s, G, k.one);
    const float2 r = make_float2(ptx::rcp_approx(den.x), ptx::rcp_approx(den.y));
    return __ffma2_rn(lap, r, c);
}
// left / right: the x neighbours of c.x / c.w (the x sums stay scalar: their operands straddle the register pairs)
template <bool PM = false>
__device__ __forceinline__ F4 update4(const F4 &c, float left, float right, const F4 &ym, const F4 &yp,
                                      const F4 &zm, const F4 &zp, const Consts &k)
{
    const float2 sx01 = make_float2(c.y + left, c.z + c.x);
    const float2 sx23 = make_float2(c.w + c.y, right + c.z);
    if (PM) {
        const float2 gx01 = make_float2(c.y - left, c.z - c.x), gx23 = make_float2(c.w - c.y, right - c.z);
        const float2 o01 = update2_pm(make_float2(c.x, c.y), sx01, gx01, make_float2(ym.x, ym.y), make_float2(yp.x, yp.y),
                                      make_float2(zm.x, zm.y), make_float2(zp.x, zp.y), k);
        const float2 o23 = update2_pm(make_float2(c.z, c.w), sx23, gx23, make_float2(ym.z, ym.w), make_float2(yp.z, yp.w),
                                      make_float2(zm.z, zm.w), make_float2(zp.z, zp.w), k);
        return F4{o01.x, o01.y, o23.x, o23.y};
    }
    const float2 o01 = update2(make_float2(c.x, c.y), sx01, make_float2(ym.x, ym.y), make_float2(yp.x, yp.y),
                               make_float2(zm.x, zm.y), make_float2(zp.x, zp.y), k);
    const float2 o23 = update2(make_float2(c.z, c.w), sx23, make_float2(ym.z, ym.w), make_float2(yp.z, yp.w),
                               make_float2(zm.z, zm.w), make_float2(zp.z, zp.w), k);
    return F4{o01.x, o01.y, o23.x, o23.y};
}

// Even reflection of a plane index about the cube faces (-1 -> 0, n -> n-1, ...).
__device__ __forceinline__ int mirror(int i, int n)
{
    const int p = 2 * n;
    int m = i % p;
    if (m < 0) m += p;
    return m < n ? m : p - 1 - m;
}

}  // namespace idg
