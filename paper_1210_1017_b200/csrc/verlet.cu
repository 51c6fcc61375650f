// a8 - system update ("the system state can be updated by numerical
// integration ... here a second-order Verlet algorithm is used"; L116: for dynamic boundary
// particles "the integration update for position and velocity is not performed").
// Formulas are reading A7 of DESIGN.md:
//   ordinary step     v+ = v(n-1) + 2 dt a,  rho+ = rho(n-1) + 2 dt drho
//   corrective step   v+ = v + dt a,         rho+ = rho + dt drho        (step 0 and every Ns-th)
//   always            r+ = r + dt v + dt^2 a / 2 ;  (v, rho)(n-1) <- (v, rho)
// The new p/rho^2 (Tait, L112) is stored with the position for the next interaction pass.
// HBM-bound: 68 B read + 48 B written per particle.  Also holds the id-order download pack.
#include "sph_internal.cuh"

namespace sph {

__global__ void __launch_bounds__(256)
verlet_kernel(uint32_t n, float4 *__restrict__ pos4, float4 *__restrict__ velrho4,
              float4 *__restrict__ velrhoM1, const float4 *__restrict__ acc4,
              const uint32_t *__restrict__ idt, uint32_t *__restrict__ flags, PhysC ph, float dt,
              int corrective)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = pos4[i];
    float4 v = velrho4[i];
    float4 m = velrhoM1[i];
    float4 a = __ldcs(acc4 + i);
    const bool fluid = (idt[i] & TYPE_BIT) == 0;
    const float dt2 = dt + dt, hdt2 = 0.5f * dt * dt;
    float rho_new = corrective ? fmaf(dt, a.w, v.w) : fmaf(dt2, a.w, m.w);
    float4 vn = v;
    if (fluid) {
        vn.x = corrective ? fmaf(dt, a.x, v.x) : fmaf(dt2, a.x, m.x);
        vn.y = corrective ? fmaf(dt, a.y, v.y) : fmaf(dt2, a.y, m.y);
        vn.z = corrective ? fmaf(dt, a.z, v.z) : fmaf(dt2, a.z, m.z);
        p.x = fmaf(hdt2, a.x, fmaf(dt, v.x, p.x));
        p.y = fmaf(hdt2, a.y, fmaf(dt, v.y, p.y));
        p.z = fmaf(hdt2, a.z, fmaf(dt, v.z, p.z));
    }
    vn.w = rho_new;
    // one test covers position, velocity, density and the rates they came from (inf - inf and 0 * inf
    // are NaN, so the sum is finite exactly when every term is)
    const float chk = (p.x + p.y + p.z) + (vn.x + vn.y + vn.z) + rho_new + (a.x + a.y + a.z + a.w);
    if (!(isfinite(chk) && rho_new > 0.f))
        atomicOr(flags, FLAG_NONFINITE);
    p.w = tait_p_over_rho2(rho_new, ph);
    pos4[i] = p;
    velrho4[i] = vn;
    velrhoM1[i] = v;
}

cudaError_t launch_verlet(sph_ctx *c, float dt, int corrective)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    verlet_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->pos4[c->cur], c->velrho4[c->cur],
                                                        c->velrhoM1[c->cur], c->acc4, c->idt[c->cur],
                                                        c->flags, c->phys, dt, corrective);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- download: scatter to id order into packed staging arrays ----------------------------------
__global__ void __launch_bounds__(256)
download_pack_kernel(uint32_t n, const float4 *__restrict__ pos4, const float4 *__restrict__ velrho4,
                     const float4 *__restrict__ acc4, const uint32_t *__restrict__ idt,
                     float *__restrict__ pos3, float *__restrict__ vel3, float *__restrict__ rho,
                     float *__restrict__ acc3, float *__restrict__ drho)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t id = idt[i] & ID_MASK;
    float4 p = pos4[i], v = velrho4[i], a = acc4[i];
    if (pos3) { pos3[3 * id] = p.x; pos3[3 * id + 1] = p.y; pos3[3 * id + 2] = p.z; }
    if (vel3) { vel3[3 * id] = v.x; vel3[3 * id + 1] = v.y; vel3[3 * id + 2] = v.z; }
    if (rho) rho[id] = v.w;
    if (acc3) { acc3[3 * id] = a.x; acc3[3 * id + 1] = a.y; acc3[3 * id + 2] = a.z; }
    if (drho) drho[id] = a.w;
}

cudaError_t launch_download_pack(sph_ctx *c, float *pos3, float *vel3, float *rho, float *acc3, float *drho)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    download_pack_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->pos4[c->cur], c->velrho4[c->cur], c->acc4,
                                                               c->idt[c->cur], pos3, vel3, rho, acc3, drho);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- exact checkpoint: the Verlet n-1 state in id order (particle data go to
// the host "only when saving"; a saved run must continue on the same trajectory) -------------------
__global__ void __launch_bounds__(256)
m1_pack_kernel(uint32_t n, const float4 *__restrict__ velrhoM1, const uint32_t *__restrict__ idt,
               float *__restrict__ vel3, float *__restrict__ rho)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t id = idt[i] & ID_MASK;
    const float4 m = velrhoM1[i];
    if (vel3) { vel3[3 * id] = m.x; vel3[3 * id + 1] = m.y; vel3[3 * id + 2] = m.z; }
    if (rho) rho[id] = m.w;
}

cudaError_t launch_m1_pack(sph_ctx *c, float *vel3, float *rho)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    m1_pack_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->velrhoM1[c->cur], c->idt[c->cur], vel3, rho);
    c->n_launches++;
    return cudaGetLastError();
}

// live arrays are in id order (right after an upload): slot i holds particle i
__global__ void __launch_bounds__(256)
m1_unpack_kernel(uint32_t n, const float *__restrict__ vel3, const float *__restrict__ rho,
                 float4 *__restrict__ velrhoM1, uint32_t *__restrict__ flags)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 m = make_float4(vel3[3 * i], vel3[3 * i + 1], vel3[3 * i + 2], rho[i]);
    if (!(isfinite(m.x + m.y + m.z + m.w) && m.w > 0.f)) atomicOr(flags, FLAG_NONFINITE);
    velrhoM1[i] = m;
}

cudaError_t launch_m1_unpack(sph_ctx *c, const float *vel3, const float *rho)
{
    uint32_t n = (uint32_t)c->n;
    if (n == 0) return cudaSuccess;
    m1_unpack_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, vel3, rho, c->velrhoM1[c->cur], c->flags);
    c->n_launches++;
    return cudaGetLastError();
}

// ---- variable time step: per-sub-domain maxima ("minimum and maximum values of certain
// physical quantities need to be found among all particles, and for this, efficient CUDA reduction
// algorithms ... are employed"; L222: every sub-domain finds its own dt_k, the step uses the minimum).
// Reading A8b: dt = cfl * min( sqrt(h / max|a|) over fluid, h / max(c_i + max_j |mu_ij|) over all ).
// Slabs are contiguous ranges of the sorted order, so a thread finds its slab in the range table; the
// maxima of non-negative floats are taken on their bit patterns (shared, then global atomicMax).
// HBM-bound: reads acc4 (16 B), rho (velrho4, 16 B), mumax (4 B), idt (4 B) per particle.
__global__ void __launch_bounds__(256)
dt_reduce_kernel(uint32_t n, const float4 *__restrict__ acc4, const float4 *__restrict__ velrho4,
                 const float *__restrict__ mumax, const uint32_t *__restrict__ idt,
                 const uint32_t *__restrict__ slab_begin, int n_slabs, PhysC ph, uint32_t *__restrict__ red)
{
    __shared__ uint32_t s_begin[SPH_MAX_SLABS + 1];
    __shared__ uint32_t s_red[2 * SPH_MAX_SLABS];
    if (threadIdx.x <= SPH_MAX_SLABS) s_begin[threadIdx.x] = threadIdx.x <= (uint32_t)n_slabs ? slab_begin[threadIdx.x] : 0xFFFFFFFFu;
    if (threadIdx.x < 2 * SPH_MAX_SLABS) s_red[threadIdx.x] = 0u;
    __syncthreads();
    // the loop bound is warp-uniform (whole warps iterate together; lanes past n are masked), because
    // the body uses full-mask warp collectives
    for (uint32_t i0 = blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < n; i0 += gridDim.x * blockDim.x) {
        const uint32_t i = i0 + (threadIdx.x & 31u);
        const bool valid = i < n;
        float sig = 0.0f, a2 = 0.0f;
        int s = 0;
        if (valid) {
            const float4 a = __ldg(acc4 + i);
            const float rho = __ldg(velrho4 + i).w;
            const bool fluid = (__ldg(idt + i) & TYPE_BIT) == 0;
            const float x = rho * ph.inv_rho0;
            const float c = ph.gamma == 7 ? ph.c0 * x * x * x : ph.c0 * __powf(x, 0.5f * (float)(ph.gamma - 1));
            sig = c + __ldg(mumax + i);
            a2 = fluid ? fmaf(a.z, a.z, fmaf(a.y, a.y, a.x * a.x)) : 0.0f;
            for (int k = 1; k < n_slabs; ++k) s += (i >= s_begin[k]) ? 1 : 0;
        }
        // warp-level pre-reduction when the whole warp sits in one slab (almost always)
        const int s0 = __shfl_sync(0xffffffffu, s, 0);
        if (__all_sync(0xffffffffu, !valid || s == s0)) {
            float ma = a2, ms = sig;
#pragma unroll
            for (int o = 16; o; o >>= 1) {
                ma = fmaxf(ma, __shfl_xor_sync(0xffffffffu, ma, o));
                ms = fmaxf(ms, __shfl_xor_sync(0xffffffffu, ms, o));
            }
            if ((threadIdx.x & 31) == 0) {
                atomicMax(&s_red[2 * s0], __float_as_uint(ma));
                atomicMax(&s_red[2 * s0 + 1], __float_as_uint(ms));
            }
        } else if (valid) {
            atomicMax(&s_red[2 * s], __float_as_uint(a2));
            atomicMax(&s_red[2 * s + 1], __float_as_uint(sig));
        }
    }
    __syncthreads();
    if (threadIdx.x < 2 * SPH_MAX_SLABS && s_red[threadIdx.x]) atomicMax(&red[threadIdx.x], s_red[threadIdx.x]);
}

cudaError_t launch_dt_reduce(sph_ctx *c)
{
    uint32_t n = (uint32_t)c->n;
    cudaError_t e = cudaMemsetAsync(c->dt_red, 0, sizeof(uint32_t) * 2 * SPH_MAX_SLABS, c->stream);
    if (e != cudaSuccess || n == 0) return e;
    uint32_t blocks = (n + 255) / 256;
    if (blocks > (uint32_t)c->num_sms * 8) blocks = (uint32_t)c->num_sms * 8;
    dt_reduce_kernel<<<blocks, 256, 0, c->stream>>>(n, c->acc4, c->velrho4[c->cur], c->mumax, c->idt[c->cur],
                                                   c->slab_begin, c->tagged_slabs.n_slabs, c->phys, c->dt_red);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
