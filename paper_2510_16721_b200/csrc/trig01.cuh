// trig01.cuh -- cos(pi x), sin(pi x) on [0, 1] without range reduction (the cosine tapers and cut-off functions of
// kernels_force.cu and kernels_dn.cu).  Each translation unit gets its own copy of the coefficient tables.
#pragma once

namespace cfn {

// cos(pi x) and sin(pi x) for x in [0, 1] (the taper variable): with y = x - 1/2, cos(pi x) = -sin(pi y) and
// sin(pi x) = cos(pi y); Taylor polynomials in y^2 to y^21 / y^22 (|pi y| <= pi/2), max abs error 3e-16 against
// long double.  About half the instructions of sincospi (no range reduction, no quadrant logic).
static __constant__ double kSinPi[11] = {3.1415926535897931, -5.1677127800499703, 2.5501640398773455, -0.59926452932079211,
                                  0.082145886611128233, -0.0073704309457143504, 0.00046630280576761255,
                                  -2.1915353447830217e-05, 7.9520540014755126e-07, -2.2948428997269873e-08,
                                  5.392664662608129e-10};
static __constant__ double kCosPi[12] = {1.0, -4.934802200544679, 4.0587121264167685, -1.3352627688545895,
                                  0.23533063035889321, -0.025806891390014061, 0.0019295743094039231,
                                  -0.0001046381049248457, 4.3030695870329473e-06, -1.3878952462213771e-07,
                                  3.6047307974625011e-09, -7.7007071306013539e-11};
__device__ __forceinline__ double cospi01(double x) {
    const double y = x - 0.5, z = y * y;
    double s = kSinPi[10];
#pragma unroll
    for (int k = 9; k >= 0; --k) s = fma(s, z, kSinPi[k]);
    return -(s * y);
}
__device__ __forceinline__ void sincospi01(double x, double &sn, double &cs) {
    const double y = x - 0.5, z = y * y;
    double s = kSinPi[10], c = kCosPi[11];
#pragma unroll
    for (int k = 9; k >= 0; --k) s = fma(s, z, kSinPi[k]);
#pragma unroll
    for (int k = 10; k >= 0; --k) c = fma(c, z, kCosPi[k]);
    cs = -(s * y);
    sn = c;
}

}  // namespace cfn
