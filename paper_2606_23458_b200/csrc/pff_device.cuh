// Device-side building blocks of libpff (sm_100a): element constitutive response, geometry loads,
// block reductions.  Formulas cite PAPER.md; they are written independently of oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "pff_internal.h"
#include "pff_tma.cuh"

namespace pff {

constexpr int kTPB = 256;  // threads per CTA of the chunk kernels
#ifndef PFF_STEP_TPB
#define PFF_STEP_TPB 256
#endif
constexpr int kStepTPB = PFF_STEP_TPB;  // threads per CTA of the explicit-step kernel (last warp = producer)

// Phase timestamps of the persistent kernels (instrumentation build only: -DPFF_TRACE, libpff_trace.so; the product
// library compiles the macro away).  Thread 0 of every CTA stores clock64 and %globaltimer into slot `slot` of its row of
// the buffer given to pff_trace_set: 256 words per CTA, [0,128) SM cycles, [128,256) nanoseconds.
#ifdef PFF_TRACE
#define PFF_TR(buf, on, slot)                                                                             \
    do {                                                                                                  \
        if ((buf) && threadIdx.x == 0 && (on)) {                                                          \
            unsigned long long gt_;                                                                       \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt_));                                        \
            (buf)[(size_t)blockIdx.x * 256 + (slot)] = clock64();                                         \
            (buf)[(size_t)blockIdx.x * 256 + 128 + (slot)] = (long long)gt_;                              \
        }                                                                                                 \
    } while (0)
#else
#define PFF_TR(buf, on, slot) do { } while (0)
#endif
constexpr int kTraceStepOffset = 256 * 1024;  // words: the step kernel's rows start here, the CG kernel's at 0

template <typename R>
struct MatC {  // material constants folded on the host
    R lam;     // lambda_PE or lambda_PS
    R mu;
    R K;       // 3-D bulk modulus
    R cz;      // eps_zz = cz * tr_2D (0 in plane strain, -nu/(1-nu) in plane stress)
    R gs;      // gamma_star (0 for vol-dev)
    R eta;
    // damage equation (Eq. 6 / Eq. 8): c_e = c0 + 2 H_e, kappa, s_e = 2 H_e - s0
    R c0, kappa, s0;
    // fracture energy (L69)
    R Gc, l0;
    int model;
};

// Host: fold the material into kernel constants (Eq. 6, Eq. 8).
template <typename R>
inline MatC<R> make_matc(const pff_material& m)
{
    MatC<R> c;
    const double mu = m.E / (2.0 * (1.0 + m.nu));
    const double lam = (m.plane == PFF_PLANE_STRESS) ? m.E * m.nu / (1.0 - m.nu * m.nu)
                                                      : m.E * m.nu / ((1.0 + m.nu) * (1.0 - 2.0 * m.nu));
    c.lam = R(lam); c.mu = R(mu); c.K = R(m.E / (3.0 * (1.0 - 2.0 * m.nu)));
    c.cz = R((m.plane == PFF_PLANE_STRESS) ? -m.nu / (1.0 - m.nu) : 0.0);
    c.gs = R(m.split == PFF_SPLIT_STARCONVEX ? m.gamma_star : 0.0);
    c.eta = R(m.eta);
    if (m.model == PFF_AT2) { c.c0 = R(m.Gc / m.l0); c.kappa = R(m.Gc * m.l0); c.s0 = R(0); }
    else { c.c0 = R(0); c.kappa = R(0.75 * m.Gc * m.l0); c.s0 = R(3.0 * m.Gc / (8.0 * m.l0)); }
    c.Gc = R(m.Gc); c.l0 = R(m.l0); c.model = m.model;
    return c;
}

template <typename R> __device__ __forceinline__ R rmax(R a, R b) { return a > b ? a : b; }
template <typename R> __device__ __forceinline__ R rmin(R a, R b) { return a < b ? a : b; }
__device__ __forceinline__ double rsqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ float rsqrt_(float x) { return sqrtf(x); }
__device__ __forceinline__ double rrsqrt_(double x) { return rsqrt(x); }
__device__ __forceinline__ float rrsqrt_(float x) { return rsqrtf(x); }
__device__ __forceinline__ double rfma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float rfma(float a, float b, float c) { return fmaf(a, b, c); }

// Element response: undegraded psi+ / psi- and degraded in-plane stress
//   sigma = g dpsi+/deps + dpsi-/deps,  g = (1 - d_e)^2 + eta (L79).
// SPLIT 1: spectral (Eq. 2) with closed-form principal strains of the 2x2 strain, eigenvector-free
//          stress  sigma+- = lam <tr>+- I + mu (s+-) I + mu (q+-) (eps - m I)/R.
// SPLIT 2/3: vol-dev (Eq. 3) / star-convex on the 3-D strain with eps_zz slaved (L85).
// SPLIT 0: isotropic (L79).
template <typename R, int SPLIT>
__device__ __forceinline__ void elem_response(const MatC<R>& m, R exx, R eyy, R exy, R g, R& psi_p, R& psi_m,
                                              R& sxx, R& syy, R& sxy)
{
    const R zero = R(0), half = R(0.5), two = R(2);
    if (SPLIT == PFF_SPLIT_SPECTRAL) {
        const R tr = exx + eyy, mean = half * tr, dd = half * (exx - eyy);
        // one reciprocal square root gives both the radius of Mohr's circle and its inverse (0 when eps = m I, R7)
        const R rad2 = dd * dd + exy * exy;
        const R inv = rad2 > zero ? rrsqrt_(rad2) : zero;
        const R rad = rad2 * inv;
        const R e1 = mean + rad, e2 = mean - rad;
        const R e1p = rmax(e1, zero), e2p = rmax(e2, zero), e1m = rmin(e1, zero), e2m = rmin(e2, zero);
        const R trp = rmax(tr, zero), trm = rmin(tr, zero);
        psi_p = half * m.lam * trp * trp + m.mu * (e1p * e1p + e2p * e2p);
        psi_m = half * m.lam * trm * trm + m.mu * (e1m * e1m + e2m * e2m);
        const R qp = (e1p - e2p) * inv, qm = (e1m - e2m) * inv;
        const R hp = m.lam * trp + m.mu * (e1p + e2p), hm = m.lam * trm + m.mu * (e1m + e2m);
        const R dev = m.mu * (g * qp + qm);  // multiplies (eps - mean I)
        const R hyd = g * hp + hm;
        sxx = hyd + dev * dd;
        syy = hyd - dev * dd;
        sxy = dev * exy;
    } else if (SPLIT == PFF_SPLIT_ISOTROPIC) {
        const R tr = exx + eyy;
        psi_p = half * m.lam * tr * tr + m.mu * (exx * exx + eyy * eyy + two * exy * exy);
        psi_m = zero;
        sxx = g * (m.lam * tr + two * m.mu * exx);
        syy = g * (m.lam * tr + two * m.mu * eyy);
        sxy = g * (two * m.mu * exy);
    } else {
        const R gs = (SPLIT == PFF_SPLIT_STARCONVEX) ? m.gs : zero;
        const R tr2 = exx + eyy, ezz = m.cz * tr2, tr3 = tr2 + ezz, third = tr3 * R(1.0 / 3.0);
        const R dxx = exx - third, dyy = eyy - third, dzz = ezz - third;
        const R e2 = dxx * dxx + dyy * dyy + dzz * dzz + two * exy * exy;
        const R trp = rmax(tr3, zero), trm = rmin(tr3, zero);
        psi_p = half * m.K * (trp * trp - gs * trm * trm) + m.mu * e2;
        psi_m = (R(1) + gs) * half * m.K * trm * trm;
        const R p = m.K * (R(1) + m.cz) * (g * (trp - gs * trm) + (R(1) + gs) * trm);
        const R tmg = two * m.mu * g;
        sxx = p + tmg * (dxx + m.cz * dzz);
        syy = p + tmg * (dyy + m.cz * dzz);
        sxy = tmg * exy;
    }
}

// Compact P1 geometry: grad phi1 = (b1, c1), grad phi2 = (b2, c2), grad phi3 = -(grad phi1 + grad phi2)
// (rows of Eq. 9 sum to zero), read as 128-bit loads.  In the chunk kernels the geometry is staged in shared
// memory by TMA: fp64 as double2 ga[EC] followed by double2 gb[EC], fp32 as float4[EC].
template <typename R> struct Geo;
template <> struct Geo<double> {
    typedef double2 Pair;  // (x, y) force pair of one element corner
    static constexpr int kArrays = 2;  // global streams: ga, gb (16 B per element each)
    static __device__ __forceinline__ void load(const void* ga, const void* gb, int e, double& b1, double& c1,
                                                double& b2, double& c2)
    {
        const double2 p = __ldg(reinterpret_cast<const double2*>(ga) + e);
        const double2 q = __ldg(reinterpret_cast<const double2*>(gb) + e);
        b1 = p.x; c1 = p.y; b2 = q.x; c2 = q.y;
    }
    static __device__ __forceinline__ void load_smem(const unsigned char* geo, int e, int EC, double& b1, double& c1,
                                                     double& b2, double& c2)
    {
        const double2* g = reinterpret_cast<const double2*>(geo);
        const double2 p = g[e], q = g[EC + e];
        b1 = p.x; c1 = p.y; b2 = q.x; c2 = q.y;
    }
    static __device__ __forceinline__ void store_global(void* ga, void* gb, int e, double v0, double v1, double v2, double v3)
    {
        reinterpret_cast<double2*>(ga)[e] = make_double2(v0, v1);
        reinterpret_cast<double2*>(gb)[e] = make_double2(v2, v3);
    }
    static __device__ __forceinline__ double2 pair(double x, double y) { return make_double2(x, y); }
    // force-pair slot idx = corner * EC + e: corners 1, 2 overwrite the element's own staged geometry, corner 3 and
    // the zero pair (idx 3 EC) live in the shared slot region
    static __device__ __forceinline__ double2* slot(unsigned char* geo, unsigned char* shared_slots, int idx, int EC)
    {
        return idx < 2 * EC ? reinterpret_cast<double2*>(geo) + idx : reinterpret_cast<double2*>(shared_slots) + (idx - 2 * EC);
    }
};
template <> struct Geo<float> {
    typedef float2 Pair;
    static constexpr int kArrays = 1;  // one float4 stream
    static __device__ __forceinline__ void load(const void* ga, const void*, int e, float& b1, float& c1,
                                                float& b2, float& c2)
    {
        const float4 p = __ldg(reinterpret_cast<const float4*>(ga) + e);
        b1 = p.x; c1 = p.y; b2 = p.z; c2 = p.w;
    }
    static __device__ __forceinline__ void load_smem(const unsigned char* geo, int e, int, float& b1, float& c1, float& b2,
                                                     float& c2)
    {
        const float4 p = reinterpret_cast<const float4*>(geo)[e];
        b1 = p.x; c1 = p.y; b2 = p.z; c2 = p.w;
    }
    static __device__ __forceinline__ void store_global(void* ga, void*, int e, float v0, float v1, float v2, float v3)
    {
        reinterpret_cast<float4*>(ga)[e] = make_float4(v0, v1, v2, v3);
    }
    static __device__ __forceinline__ float2 pair(float x, float y) { return make_float2(x, y); }
    static __device__ __forceinline__ float2* slot(unsigned char*, unsigned char* shared_slots, int idx, int)
    {
        return reinterpret_cast<float2*>(shared_slots) + idx;
    }
};

// element operator q^e = (c_e M^e + kappa K^e) p^e with M^e = A (1 + delta_ij) / 12 (L185), from the geometry
template <typename R>
__device__ __forceinline__ void elem_damage_apply(const MatC<R>& mat, R b1, R c1, R b2, R c2, R A, R He, R p1, R p2, R p3,
                                                  R& q1, R& q2, R& q3)
{
    const R ce = mat.c0 + R(2) * He;  // reaction coefficient (Eq. 6 / Eq. 8)
    const R m12 = ce * A * R(1.0 / 12.0), sum = p1 + p2 + p3;
    const R gx = b1 * (p1 - p3) + b2 * (p2 - p3), gy = c1 * (p1 - p3) + c2 * (p2 - p3);
    const R kA = mat.kappa * A;
    const R k1 = kA * (b1 * gx + c1 * gy), k2 = kA * (b2 * gx + c2 * gy);
    q1 = m12 * (p1 + sum) + k1;
    q2 = m12 * (p2 + sum) + k2;
    q3 = m12 * (p3 + sum) - (k1 + k2);
}

// The same operator from its 4 coefficients (what the CG iterations stream instead of geometry + area + H):
// m = c_e A / 12 and the edge weights w_ij = -kappa A grad phi_i . grad phi_j of the P1 stiffness (rows sum to zero,
// so K^e p = sum_j w_ij (p_i - p_j)).
template <typename R>
__device__ __forceinline__ void elem_coefficients(const MatC<R>& mat, R b1, R c1, R b2, R c2, R A, R He, R& m, R& w12, R& w13,
                                                  R& w23)
{
    const R kA = mat.kappa * A;
    m = (mat.c0 + R(2) * He) * A * R(1.0 / 12.0);
    w12 = -kA * (b1 * b2 + c1 * c2);
    w13 = kA * (b1 * (b1 + b2) + c1 * (c1 + c2));
    w23 = kA * (b2 * (b1 + b2) + c2 * (c1 + c2));
}

// Ordered sum of one interface node's per-chunk partials: kIfaceWidth fixed slots (unused ones hold zero) and,
// on irregular meshes only, its overflow slots.  No index has to be loaded first on regular meshes.
template <typename R>
__device__ __forceinline__ R iface_sum(const R* plane, int s, int N_sh, int n_ovf, const int32_t* ovf_rowptr)
{
    const R* hp = plane + (size_t)kIfaceWidth * s;
    R v;
    if ((reinterpret_cast<uintptr_t>(hp) & 15) == 0) {  // the usual case: the four slots in one or two 16-byte loads
        if (sizeof(R) == 8) {
            const double2 lo = reinterpret_cast<const double2*>(hp)[0], hi = reinterpret_cast<const double2*>(hp)[1];
            v = R(((lo.x + lo.y) + hi.x) + hi.y);
        } else {
            const float4 q = *reinterpret_cast<const float4*>(hp);
            v = R(((q.x + q.y) + q.z) + q.w);
        }
    } else {
        v = ((hp[0] + hp[1]) + hp[2]) + hp[3];
    }
    if (n_ovf > 0)
        for (int k = ovf_rowptr[s]; k < ovf_rowptr[s + 1]; ++k) v += plane[(size_t)kIfaceWidth * N_sh + k];
    return v;
}

// Deterministic block sum in fp64 (fixed shuffle tree, fixed warp order); result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double* s_red /* >= 32 doubles */)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) s_red[w] = v;
    __syncthreads();
    double t = 0.0;
    if (w == 0) {
        t = l < nw ? s_red[l] : 0.0;
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;
}
__device__ __forceinline__ double block_min(double v, double* s_red)
{
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) s_red[w] = v;
    __syncthreads();
    double t = INFINITY;
    if (w == 0) {
        t = l < nw ? s_red[l] : INFINITY;
        for (int o = 16; o > 0; o >>= 1) t = fmin(t, __shfl_xor_sync(0xffffffffu, t, o));
    }
    return t;
}

constexpr int kRedWarps = 16;  // warps per CTA the block reductions provide for (scratch: kCh x kRedWarps doubles)
static_assert(kTPB <= 32 * kRedWarps && kStepTPB <= 32 * kRedWarps, "block reduction scratch too small");
constexpr int kCh = 8;  // partial-sum channels of the CG kernels: p.q, r.z, r.r, z.q, q.Dinv.q, r.q, q.q, min step bound

// true in every thread of the LAST CTA of the grid to get here (self-resetting ticket); its reads that follow see every
// other CTA's earlier global writes
__device__ __forceinline__ bool last_block(unsigned int* ticket)
{
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) *ticket = 0u;
    }
    __syncthreads();
    if (s_last) __threadfence();
    return s_last;
}

// Deterministic block reduction of kCh values at once (channels 0..6 summed, channel 7 minimised): fixed
// shuffle tree, fixed warp order, two barriers.  Results land in s_out[0..kCh) (visible after the call).
__device__ __forceinline__ void block_reduce_ch(double v[kCh], double* s_w /* [kCh][kRedWarps] */, double* s_out /* [kCh] */)
{
#pragma unroll
    for (int c = 0; c < kCh; ++c)
        for (int o = 16; o > 0; o >>= 1) {
            const double t = __shfl_xor_sync(0xffffffffu, v[c], o);
            v[c] = (c == kCh - 1) ? fmin(v[c], t) : v[c] + t;
        }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) {
#pragma unroll
        for (int c = 0; c < kCh; ++c) s_w[c * kRedWarps + w] = v[c];
    }
    __syncthreads();
    if (w < kCh) {  // warp c reduces channel c
        double t = l < nw ? s_w[w * kRedWarps + l] : (w == kCh - 1 ? INFINITY : 0.0);
        for (int o = 16; o > 0; o >>= 1) {
            const double u = __shfl_xor_sync(0xffffffffu, t, o);
            t = (w == kCh - 1) ? fmin(t, u) : t + u;
        }
        if (l == 0) s_out[w] = t;
    }
    __syncthreads();
}

}  // namespace pff
