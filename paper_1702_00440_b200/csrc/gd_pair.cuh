// gd_pair.cuh -- the pair term of the softened force/jerk sums (Eq. 3, jerk sign per fn. 11 P:188), shared by
// the force kernels (gd_force.cu) and the persistent block-step loop (gd_loop.cu).  Not shared with oracle/.
#pragma once
#include "gd_common.cuh"

// ---------------------------------------------------------------------------------------------------------
// q = s^(-1/2): MUFU.RSQ64H seed (relative error ~2^-21: it sees the upper 32 bits of s only) followed by one
// third-order step  y <- y + y e (1/2 + 3/8 e),  e = 1 - s y^2   (error 5/16 e^3 ~ 2^-60: below 1 ulp).
// EPS0 = true (eps == 0): s == 0 for coincident particles and the self pair, masked to q = 0.  With eps > 0, s >= eps^2
// is a normal number and the mask is compiled out (the host picks EPS0 whenever eps^2 is zero or denormal).
template <bool EPS0>
__device__ __forceinline__ double gd_rsqrt(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    if (EPS0) {
        if (__double2hiint(s) == 0) y = 0.0;                     // contribute nothing instead of inf * 0
    }
    double t = s * y;
    double e = fma(-t, y, 1.0);
    double p = fma(0.375, e, 0.5);
    double g = y * e;
    return fma(g, p, y);
}

struct gd_src { double x, y, z, m, vx, vy, vz; };
struct gd_acc { double ax, ay, az, jx, jy, jz; };

template <bool EPS0>
__device__ __forceinline__ void gd_pair(const gd_src &i, const gd_src &j, double eps2, gd_acc &o)
{
    double rx = j.x - i.x, ry = j.y - i.y, rz = j.z - i.z;
    double wx = j.vx - i.vx, wy = j.vy - i.vy, wz = j.vz - i.vz;
    double s = fma(rx, rx, fma(ry, ry, fma(rz, rz, eps2)));
    double rw = fma(rx, wx, fma(ry, wy, rz * wz));
    double q = gd_rsqrt<EPS0>(s);
    double q2 = q * q;
    double mq3 = (j.m * q) * q2;
    double b3 = -3.0 * (rw * q2);
    o.ax = fma(mq3, rx, o.ax);
    o.ay = fma(mq3, ry, o.ay);
    o.az = fma(mq3, rz, o.az);
    o.jx = fma(mq3, fma(b3, rx, wx), o.jx);
    o.jy = fma(mq3, fma(b3, ry, wy), o.jy);
    o.jz = fma(mq3, fma(b3, rz, wz), o.jz);
}

__device__ __forceinline__ gd_src gd_load_sink(const gd_dev &d, int32_t i)
{
    double2 xy = __ldg(d.pxy + i), zm = __ldg(d.pzm + i), vxy = __ldg(d.vxy + i);
    double vz = __ldg(d.vz + i);
    return gd_src{xy.x, xy.y, zm.x, zm.y, vxy.x, vxy.y, vz};
}
