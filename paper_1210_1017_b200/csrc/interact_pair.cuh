// Pair term of the SPH interaction (Eq. (7), Eq. (9) L106 in the p/rho^2 form of DESIGN.md
// reading A2, artificial viscosity and Tait equation of state L112), scalar fp32 form, shared by the
// cross-check kernels of interact.cu and used as the model for the packed form in interact_mma.cu.
#pragma once
#include "sph_internal.cuh"

namespace sph {

// ---- pair term ---------------------------------------------------------------------------------
__device__ __forceinline__ float rsqrt_fast(float x)        // 1 MUFU, |rel err| <= 2^-22
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x)          // 1 MUFU, |rel err| <= 2^-23
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Returns F with grad_i W_ij = F r_ij, for 0 < r2 (F -> 0 smoothly at r = 2h and is clamped to
// 0 beyond, so a filter that lets a pair marginally outside 2h through changes nothing).
template <int KERNEL>
__device__ __forceinline__ float kernel_F(float r2, const PhysC &ph)
{
    float rinv = rsqrt_fast(r2);
    float r = r2 * rinv;
    if (KERNEL == 0) {                      // Wendland C2: F = -5 aD (1 - q/2)^3 / h^2
        float t = fmaxf(fmaf(-ph.inv_h_half, r, 1.0f), 0.0f);
        return ph.kF * t * t * t;
    } else {                                // cubic spline, kF = aD / h^2
        float q = r * (2.0f * ph.inv_h_half);
        float t = fmaxf(2.0f - q, 0.0f);
        float f = q <= 1.0f ? fmaf(2.25f, q, -3.0f) : -0.75f * t * t * rinv * ph.h;
        return ph.kF * f;
    }
}

template <bool GAMMA7>
__device__ __forceinline__ float sound_speed(float rho, const PhysC &ph)
{
    float x = rho * ph.inv_rho0;
    if (GAMMA7) return ph.c0 * x * x * x;               // c0 (rho/rho0)^((gamma-1)/2), gamma = 7
    return ph.c0 * __powf(x, 0.5f * (float)(ph.gamma - 1));
}

// Adds the contribution of neighbour j to (ax, ay, az, dr); masses are applied by the caller
// (mj = 1 in the uniform-mass path).  Branch-free: the viscous term uses min(v_ij.r_ij, 0).
// MU: also track max_j |mu_ij| (variable time step, reading A8b) over the pairs with
// r < 2h exactly (|mu| does not vanish at the edge of the support, unlike F) and mj != 0.
template <int KERNEL, bool GAMMA7, bool MU>
__device__ __forceinline__ void pair_term(float dx, float dy, float dz, float r2,
                                          float vxi, float vyi, float vzi, float rhoi, float Pi_, float ci,
                                          float4 vj, float Pj, float mj, const PhysC &ph,
                                          float &ax, float &ay, float &az, float &dr, float &mumax)
{
    float F = kernel_F<KERNEL>(r2, ph) * mj;
    float dvx = vxi - vj.x, dvy = vyi - vj.y, dvz = vzi - vj.z;
    float dot = fmaf(dvz, dz, fmaf(dvy, dy, dvx * dx));
    dr = fmaf(F, dot, dr);                                            // Eq. (7)
    // L112: Pi = -alpha cbar mu / rhobar = -alpha h (ci+cj) dot / ((r2+eta2)(rhoi+rhoj)) if dot < 0
    float cj = sound_speed<GAMMA7>(vj.w, ph);
    const float rsum = rhoi + vj.w;
    const float rc = rcp_fast((r2 + ph.eta2) * rsum);
    float visc = -ph.alpha_h * (ci + cj) * fminf(dot, 0.0f) * rc;
    if (MU) {
        const float mu = ph.h * fabsf(dot) * (rc * rsum);             // h |v_ij.r_ij| / (r2 + eta2)
        mumax = fmaxf(mumax, (r2 < ph.four_h2 && mj != 0.0f) ? mu : 0.0f);
    }
    float coef = -F * (Pi_ + Pj + visc);                              // Eq. (9)
    ax = fmaf(coef, dx, ax);
    ay = fmaf(coef, dy, ay);
    az = fmaf(coef, dz, az);
}

}  // namespace sph
