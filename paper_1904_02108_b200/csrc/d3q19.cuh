// D3Q19 lattice constants and the fp32 BGK collision with body force, in deviation form.
//
// Populations are stored as  df_i = f_i - t_i: the rest state is all
// zeros and the O(1) part of rho never enters an fp32 sum.
//
// Direction numbering is lexicographic in (ez, ey, ex) over the 19 vectors with |e|^2 <= 2, so
// that the opposite of direction i is 18 - i and i = 9 is the rest population (P:35 gives no
// order; it is internal and never visible at the ABI, reading R2).
#pragma once
#include <cuda_runtime.h>

namespace lbmk {

constexpr int NQ = 19;

// e_i as constexpr functions (folded to literals once the direction loops are unrolled).
__host__ __device__ constexpr int dir_ez(int i) { return i < 5 ? -1 : (i < 14 ? 0 : 1); }
__host__ __device__ constexpr int dir_ey(int i)
{
    return i < 5 ? (i == 0 ? -1 : (i == 4 ? 1 : 0)) : (i < 14 ? ((i - 5) / 3 - 1) : (i == 14 ? -1 : (i == 18 ? 1 : 0)));
}
__host__ __device__ constexpr int dir_ex(int i)
{
    return i < 5 ? (i == 1 ? -1 : (i == 3 ? 1 : 0)) : (i < 14 ? ((i - 5) % 3 - 1) : (i == 15 ? -1 : (i == 17 ? 1 : 0)));
}
__host__ __device__ constexpr int dir_opp(int i) { return NQ - 1 - i; }
__host__ __device__ constexpr int dir_norm2(int i)
{
    return dir_ex(i) * dir_ex(i) + dir_ey(i) * dir_ey(i) + dir_ez(i) * dir_ez(i);
}
// t_i: 1/3 (rest), 1/18 (axis), 1/36 (face diagonal); c_s^2 = 1/3.
__host__ __device__ constexpr float dir_weight(int i)
{
    return dir_norm2(i) == 0 ? (1.0f / 3.0f) : (dir_norm2(i) == 1 ? (1.0f / 18.0f) : (1.0f / 36.0f));
}

// Relaxation and forcing constants, filled on the host from the double-precision tau.
struct CollisionConst {
    float omega;       // 1/tau
    float keep;        // 1 - 1/tau
    float guo;         // 1 - 1/(2 tau)
    float tau;
    float gbx, gby, gbz;  // uniform body acceleration
    int shift_forcing;    // 0: Guo source term (R3); 1: paper's U + tau*a shift
};

// Moments of eq. (1), from deviations: rho = 1 + sum df, rho U = sum e_i df (sum e_i t_i = 0).
__device__ __forceinline__ void moments(const float (&df)[NQ], float &drho, float &ux, float &uy, float &uz)
{
    float s = 0.f, jx = 0.f, jy = 0.f, jz = 0.f;
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        s += df[i];
        if (dir_ex(i) == 1) jx += df[i];
        if (dir_ex(i) == -1) jx -= df[i];
        if (dir_ey(i) == 1) jy += df[i];
        if (dir_ey(i) == -1) jy -= df[i];
        if (dir_ez(i) == 1) jz += df[i];
        if (dir_ez(i) == -1) jz -= df[i];
    }
    const float inv = __fdividef(1.0f, 1.0f + s);   // MUFU.RCP, relative error < 2^-22
    drho = s;
    ux = jx * inv;
    uy = jy * inv;
    uz = jz * inv;
}

// BGK collision, eq. (2),(3) (rho per R1), with acceleration a = G + g_body (R4):
//   Guo (R3):   u* = U + a/2,  f_i <- f_i - (f_i - Eq_i(rho,u*))/tau
//                                       + (1 - 1/(2tau)) t_i rho [3 (e_i - u*).a + 9 (e_i.u*)(e_i.a)]
//   shift:  f_i <- f_i - (f_i - Eq_i(rho, U + tau a))/tau
// all in deviation form: Eq_i - t_i = t_i [drho + rho (3 e.u + 4.5 (e.u)^2 - 1.5 u.u)].
__device__ __forceinline__ void collide(float (&df)[NQ], float ax, float ay, float az, const CollisionConst &c)
{
    float drho, ux, uy, uz;
    moments(df, drho, ux, uy, uz);
    const float rho = 1.0f + drho;
    const float h = c.shift_forcing ? c.tau : 0.5f;
    const float vx = fmaf(h, ax, ux), vy = fmaf(h, ay, uy), vz = fmaf(h, az, uz);
    // The update of direction i splits into a part even in e_i and a part odd in e_i, shared by the
    // pair (i, opp i) = (i, 18 - i).  With A = rho/tau, B = (1 - 1/(2 tau)) rho (B = 0 for the shift):
    //   even_i = t_i [ drho/tau - 1.5 A v.v - 3 B v.a + (e.v) (e.(4.5 A v + 9 B a)) ]
    //   odd_i  = t_i  e.(3 A v + 3 B a)
    //   f_i <- keep f_i + even_i + odd_i,   f_opp <- keep f_opp + even_i - odd_i
    const float A = c.omega * rho;
    const float B = c.shift_forcing ? 0.0f : c.guo * rho;
    const float c0 = fmaf(c.omega, drho, -(1.5f * A * (vx * vx + vy * vy + vz * vz) + 3.0f * B * (vx * ax + vy * ay + vz * az)));
    const float qx = fmaf(4.5f * A, vx, 9.0f * B * ax), qy = fmaf(4.5f * A, vy, 9.0f * B * ay), qz = fmaf(4.5f * A, vz, 9.0f * B * az);
    const float px = 3.0f * fmaf(A, vx, B * ax), py = 3.0f * fmaf(A, vy, B * ay), pz = 3.0f * fmaf(A, vz, B * az);
    df[9] = fmaf(c.keep, df[9], dir_weight(9) * c0);
#pragma unroll
    for (int i = 0; i < 9; ++i) {
        const float w = dir_weight(i);
        const float ev = dir_ex(i) * vx + dir_ey(i) * vy + dir_ez(i) * vz;
        const float eq = dir_ex(i) * qx + dir_ey(i) * qy + dir_ez(i) * qz;
        const float ep = dir_ex(i) * px + dir_ey(i) * py + dir_ez(i) * pz;
        const float even = w * fmaf(ev, eq, c0);
        const float odd = w * ep;
        df[i] = fmaf(c.keep, df[i], even + odd);
        df[dir_opp(i)] = fmaf(c.keep, df[dir_opp(i)], even - odd);
    }
}

// Eq_i(rho, u) - t_i, used by lbm_set_fields (R18).
__device__ __forceinline__ float equilibrium_dev(int i, float drho, float ux, float uy, float uz)
{
    const float eu = dir_ex(i) * ux + dir_ey(i) * uy + dir_ez(i) * uz;
    const float uu15 = 1.5f * (ux * ux + uy * uy + uz * uz);
    return dir_weight(i) * fmaf(1.0f + drho, fmaf(eu, fmaf(4.5f, eu, 3.0f), -uu15), drho);
}

}  // namespace lbmk
