// md_pair.cuh -- device helpers and the pair functions (S:O1-O4) shared by the force kernels of md_forces.cu
// (L2-resident gathers) and md_staged.cu (shared-memory staged neighbourhoods).  Product code: nothing here is
// shared with oracle/.
#pragma once
#include "md_internal.cuh"

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void red_add_v4(float4* addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void red_add_f32(float* addr, float a) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(a) : "memory");
}
__device__ __forceinline__ float4 ldg4(const float4* p) { return __ldg(p); }

// S:H9 robust fp32 minimum image: subtract L from the larger coordinate before differencing (both inner
// subtractions are exact), used only by warps that hold a pair crossing a periodic face.
__device__ __forceinline__ float min_image(float xj, float xi, float L, float hL) {
    float t = xj - xi;
    if (t > hL) t = (xj - L) - xi;
    else if (t < -hL) t = xj - (xi - L);
    return t;
}

// S:O0 / S:Q5 predicate in fp64, fixed operation order, no FMA contraction.
static __device__ __noinline__ bool inside_fp64(float4 xi, float4 xj, double Lx, double Ly, double Lz, double thr2) {
    double dx = (double)xj.x - (double)xi.x;
    if (dx > 0.5 * Lx) dx -= Lx; else if (dx < -0.5 * Lx) dx += Lx;
    double dy = (double)xj.y - (double)xi.y;
    if (dy > 0.5 * Ly) dy -= Ly; else if (dy < -0.5 * Ly) dy += Ly;
    double dz = (double)xj.z - (double)xi.z;
    if (dz > 0.5 * Lz) dz -= Lz; else if (dz < -0.5 * Lz) dz += Lz;
    double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    return d2 < thr2;
}

// in-cutoff decision: fp32 away from the threshold, fp64 inside the band
__device__ __forceinline__ bool in_cutoff(const DevParams& P, float d2, float4 xi, float4 xj) {
    const float t = d2 - P.rc2;
    bool in = t < 0.0f;
    if (fabsf(t) < P.band_abs) in = inside_fp64(xi, xj, P.dLx, P.dLy, P.dLz, P.rc2d);
    return in;
}

// ------------------------------------------------------------------------------------------------
// pair functions.  d = r_j - r_i (minimum image).  They return the force ON j:  F_j = g*d (+ ...),
// F_i = -F_j, and the pair energy V; the callers split V in halves (S:O1).
// ------------------------------------------------------------------------------------------------
// O1 Eq.(1), cut + energy shift P:99;  O2 WCA is the same with rc = 2^(1/6) sigma, V_c = -eps.
__device__ __forceinline__ void lj_pair(const DevParams& P, float d2, float& g, float& V) {
    float inv = rcp_approx(d2);
    float inv3 = inv * inv * inv;
    g = inv * inv3 * fmaf(P.lj_a, inv3, -P.lj_b);            // 24 eps s6 (2 s6 - 1) / d2, s6 = sigma^6 / d2^3
    V = fmaf(inv3, fmaf(P.lj_c, inv3, -P.lj_d), -P.vshift);   // 4 eps s6 (s6 - 1) - V_c
}

struct Rot { float m[3][3]; };
__device__ __forceinline__ Rot quat_to_rot(float4 q) {   // q = (w,x,y,z) stored as (.x,.y,.z,.w) = (w,x,y,z)
    float w = q.x, x = q.y, y = q.z, z = q.w;
    Rot R;
    R.m[0][0] = 1.f - 2.f * (y * y + z * z); R.m[0][1] = 2.f * (x * y - w * z);       R.m[0][2] = 2.f * (x * z + w * y);
    R.m[1][0] = 2.f * (x * y + w * z);       R.m[1][1] = 1.f - 2.f * (x * x + z * z); R.m[1][2] = 2.f * (y * z - w * x);
    R.m[2][0] = 2.f * (x * z - w * y);       R.m[2][1] = 2.f * (y * z + w * x);       R.m[2][2] = 1.f - 2.f * (x * x + y * y);
    return R;
}

// angular factor of one particle (S:O4, factorised form): with v = R^T * dir (dir = +u for i, -u for j)
//   A = sum_a exp((b_a.v - 1)/w^2),   S = (1/w^2) R sum_a e_a b_a
// NP = number of patches known at compile time (4: the tetrahedral model of config 4, fully unrolled), 0 = P.n_patches
template <int NP>
__device__ __forceinline__ void patch_factor(const DevParams& P, const Rot& R, float ux, float uy, float uz,
                                             float& A, float& Sx, float& Sy, float& Sz) {
    float vx = R.m[0][0] * ux + R.m[1][0] * uy + R.m[2][0] * uz;
    float vy = R.m[0][1] * ux + R.m[1][1] * uy + R.m[2][1] * uz;
    float vz = R.m[0][2] * ux + R.m[1][2] * uy + R.m[2][2] * uz;
    const float k = P.inv_w2 * 1.4426950408889634f;   // exp(x) = 2^(x log2 e)
    float a = 0.f, bx = 0.f, by = 0.f, bz = 0.f;
    const int np = NP > 0 ? NP : P.n_patches;
#pragma unroll
    for (int p = 0; p < np; ++p) {
        float c = P.pdir[p][0] * vx + P.pdir[p][1] * vy + P.pdir[p][2] * vz;
        float e = ex2_approx((c - 1.0f) * k);
        a += e;
        bx = fmaf(e, P.pdir[p][0], bx); by = fmaf(e, P.pdir[p][1], by); bz = fmaf(e, P.pdir[p][2], bz);
    }
    A = a;
    Sx = P.inv_w2 * (R.m[0][0] * bx + R.m[0][1] * by + R.m[0][2] * bz);
    Sy = P.inv_w2 * (R.m[1][0] * bx + R.m[1][1] * by + R.m[1][2] * bz);
    Sz = P.inv_w2 * (R.m[2][0] * bx + R.m[2][1] * by + R.m[2][2] * bz);
}

// Both angular factors of a pair at once for the TETRAHEDRAL patch set of config 4 (B:10, S:O4: b_a = (+-1, +-1, +-1)/sqrt(3)
// with an even number of minus signs), in packed f32x2: .x = particle i (direction +u), .y = particle j (direction -u).
// The four dot products b_a.v need no multiplications (sums and differences of the components of v), and neither does
// sum_a e_a b_a; 1/sqrt(3) is folded into the exponent scale and into the prefactor of S.  ~28 packed instructions + 8 MUFU
// for both particles, against 2 x 45 scalar ones in patch_factor<4>.  R2[m][n] = (R_i[m][n], R_j[m][n]).
__device__ __forceinline__ void patch_factor2_tetra(const DevParams& P, const float2 (&R2)[3][3], float ux, float uy, float uz,
                                                    float2& A, float2& Sx, float2& Sy, float2& Sz) {
    const float2 U0 = make_float2(ux, -ux), U1 = make_float2(uy, -uy), U2 = make_float2(uz, -uz);
    // v = R^T dir
    const float2 vx = __ffma2_rn(R2[2][0], U2, __ffma2_rn(R2[1][0], U1, __fmul2_rn(R2[0][0], U0)));
    const float2 vy = __ffma2_rn(R2[2][1], U2, __ffma2_rn(R2[1][1], U1, __fmul2_rn(R2[0][1], U0)));
    const float2 vz = __ffma2_rn(R2[2][2], U2, __ffma2_rn(R2[1][2], U1, __fmul2_rn(R2[0][2], U0)));
    const float2 nvz = make_float2(-vz.x, -vz.y);
    const float2 s = __fadd2_rn(vx, vy), d = __fadd2_rn(vx, make_float2(-vy.x, -vy.y));
    // sqrt(3) b_a . v for b_1 = (1,1,1), b_2 = (1,-1,-1), b_3 = (-1,1,-1), b_4 = (-1,-1,1)
    const float2 c1 = __fadd2_rn(s, vz), c2 = __fadd2_rn(d, nvz), c3 = __fadd2_rn(make_float2(-d.x, -d.y), nvz),
                 c4 = __fadd2_rn(vz, make_float2(-s.x, -s.y));
    const float k = P.inv_w2 * 1.4426950408889634f;                 // exp(x) = 2^(x log2 e)
    const float2 ks = make_float2(k * 0.57735026918962576f, k * 0.57735026918962576f), nk = make_float2(-k, -k);
    const float2 x1 = __ffma2_rn(c1, ks, nk), x2 = __ffma2_rn(c2, ks, nk), x3 = __ffma2_rn(c3, ks, nk), x4 = __ffma2_rn(c4, ks, nk);
    const float2 e1 = make_float2(ex2_approx(x1.x), ex2_approx(x1.y)), e2 = make_float2(ex2_approx(x2.x), ex2_approx(x2.y));
    const float2 e3 = make_float2(ex2_approx(x3.x), ex2_approx(x3.y)), e4 = make_float2(ex2_approx(x4.x), ex2_approx(x4.y));
    const float2 p12 = __fadd2_rn(e1, e2), p34 = __fadd2_rn(e3, e4);
    const float2 m12 = __fadd2_rn(e1, make_float2(-e2.x, -e2.y)), m34 = __fadd2_rn(e3, make_float2(-e4.x, -e4.y));
    A = __fadd2_rn(p12, p34);
    // sqrt(3) sum_a e_a b_a = (e1 + e2 - e3 - e4, e1 - e2 + e3 - e4, e1 - e2 - e3 + e4)
    const float2 bx = __fadd2_rn(p12, make_float2(-p34.x, -p34.y)), by = __fadd2_rn(m12, m34), bz = __fadd2_rn(m12, make_float2(-m34.x, -m34.y));
    const float w = P.inv_w2 * 0.57735026918962576f;
    const float2 w2 = make_float2(w, w);
    Sx = __fmul2_rn(w2, __ffma2_rn(R2[0][2], bz, __ffma2_rn(R2[0][1], by, __fmul2_rn(R2[0][0], bx))));
    Sy = __fmul2_rn(w2, __ffma2_rn(R2[1][2], bz, __ffma2_rn(R2[1][1], by, __fmul2_rn(R2[1][0], bx))));
    Sz = __fmul2_rn(w2, __ffma2_rn(R2[2][2], bz, __ffma2_rn(R2[2][1], by, __fmul2_rn(R2[2][0], bx))));
}

// x^n for a small runtime integer n >= 1 by squaring (the paper's exponents: 100 = 200/2 and 5 = 10/2)
__device__ __forceinline__ float ipow(float x, int n) {
    float r = 1.0f;
    while (n) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}

// The paper's own patchy model, Eqs. (2)-(4) P:103-113 under reading S:Q1 (S:8(f2)): core eps (sigma/r)^m plus, for every
// patch pair (a of i, b of j) closer than rcut_patch, -eps_p exp[-1/2 (r_ab / w)^n] with r_ab the patch-patch distance,
// patches at pp_radius * R dir from the centres.  With e = d + p_b - p_a, u2 = |e|^2, g = 1/2 (u2 / w^2)^(n/2):
//   term = -eps_p exp(-g),  d term / d e = c e,  c = -term n g / u2;  F_j = -sum c e,  tau_i = sum p_a x (c e),  tau_j = -sum p_b x (c e)
template <bool NEED_TJ>
__device__ __forceinline__ void patchy_pp_pair(const DevParams& P, float dx, float dy, float dz, float d2, const Rot& Ri, float4 qj,
                                               float& fx, float& fy, float& fz, float& V,
                                               float& tix, float& tiy, float& tiz, float& tjx, float& tjy, float& tjz) {
    const Rot Rj = quat_to_rot(qj);
    const float inv = 1.0f / d2;
    V = P.eps * ipow(P.sig2 * inv, P.pp_core_half);          // Eq. (3)
    const float gc = P.pp_core_n * V * inv;                   // F_j = -dV/dr_vec = m V r_vec / r^2
    fx = gc * dx; fy = gc * dy; fz = gc * dz;
    tix = tiy = tiz = 0.f;
    tjx = tjy = tjz = 0.f;
    for (int a = 0; a < P.n_patches; ++a) {
        const float pax = P.pp_radius * (Ri.m[0][0] * P.pdir[a][0] + Ri.m[0][1] * P.pdir[a][1] + Ri.m[0][2] * P.pdir[a][2]);
        const float pay = P.pp_radius * (Ri.m[1][0] * P.pdir[a][0] + Ri.m[1][1] * P.pdir[a][1] + Ri.m[1][2] * P.pdir[a][2]);
        const float paz = P.pp_radius * (Ri.m[2][0] * P.pdir[a][0] + Ri.m[2][1] * P.pdir[a][1] + Ri.m[2][2] * P.pdir[a][2]);
        for (int b = 0; b < P.n_patches; ++b) {
            const float pbx = P.pp_radius * (Rj.m[0][0] * P.pdir[b][0] + Rj.m[0][1] * P.pdir[b][1] + Rj.m[0][2] * P.pdir[b][2]);
            const float pby = P.pp_radius * (Rj.m[1][0] * P.pdir[b][0] + Rj.m[1][1] * P.pdir[b][1] + Rj.m[1][2] * P.pdir[b][2]);
            const float pbz = P.pp_radius * (Rj.m[2][0] * P.pdir[b][0] + Rj.m[2][1] * P.pdir[b][1] + Rj.m[2][2] * P.pdir[b][2]);
            const float ex = (dx + pbx) - pax, ey = (dy + pby) - pay, ez = (dz + pbz) - paz;
            const float u2 = fmaf(ez, ez, fmaf(ey, ey, ex * ex));
            if (!(u2 < P.pp_rc2)) continue;                   // only patch pairs closer than 0.18 sigma
            const float g = 0.5f * ipow(u2 * P.pp_inv_w2, P.pp_half_n);
            const float term = -P.eps_patch * ex2_approx(-g * 1.4426950408889634f);   // Eq. (4), one patch pair
            V += term;
            if (u2 > 0.0f) {
                const float c = -term * P.pp_n * g / u2;
                const float gx = c * ex, gy = c * ey, gz = c * ez;
                fx -= gx; fy -= gy; fz -= gz;
                tix += pay * gz - paz * gy; tiy += paz * gx - pax * gz; tiz += pax * gy - pay * gx;
                if (NEED_TJ) { tjx -= pby * gz - pbz * gy; tjy -= pbz * gx - pbx * gz; tjz -= pbx * gy - pby * gx; }
            }
        }
    }
}

// O4 (B:10): WCA core + patch term.  Outputs force on j (fx,fy,fz), V, torque on i, torque on j.
// Ri = rotation matrix of particle i (callers that keep i fixed over a loop compute it once).
template <bool NEED_TJ, int NP>
__device__ __forceinline__ void patchy_pair(const DevParams& P, float dx, float dy, float dz, float d2, const Rot& Ri, float4 qj,
                                            float& fx, float& fy, float& fz, float& V,
                                            float& tix, float& tiy, float& tiz, float& tjx, float& tjy, float& tjz) {
    float rinv = rsqrt_approx(d2);
    float r = d2 * rinv;
    float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
    float Ai, Six, Siy, Siz, Aj, Sjx, Sjy, Sjz;
    const Rot Rj = quat_to_rot(qj);
    if (NP == 4 && P.tetra) {       // config 4's tetrahedral patch set: both factors in packed f32x2
        float2 R2[3][3];
#pragma unroll
        for (int m = 0; m < 3; ++m)
#pragma unroll
            for (int n = 0; n < 3; ++n) R2[m][n] = make_float2(Ri.m[m][n], Rj.m[m][n]);
        float2 A, Sx, Sy, Sz;
        patch_factor2_tetra(P, R2, ux, uy, uz, A, Sx, Sy, Sz);
        Ai = A.x; Aj = A.y; Six = Sx.x; Sjx = Sx.y; Siy = Sy.x; Sjy = Sy.y; Siz = Sz.x; Sjz = Sz.y;
    } else {
        patch_factor<NP>(P, Ri, ux, uy, uz, Ai, Six, Siy, Siz);
        patch_factor<NP>(P, Rj, -ux, -uy, -uz, Aj, Sjx, Sjy, Sjz);
    }
    float dr = r - P.sigma;
    float G = ex2_approx(-dr * dr * P.inv_2sr2 * 1.4426950408889634f);
    float dG = -dr * P.inv_sr2 * G;
    float eG = P.eps_patch * G;
    V = -eG * Ai * Aj;
    // dA_i/dr_vec = (S_i - (S_i.u)u)/r ; dA_j/dr_vec = -(S_j - (S_j.u)u)/r
    float siu = Six * ux + Siy * uy + Siz * uz;
    float sju = Sjx * ux + Sjy * uy + Sjz * uz;
    float ci = eG * Aj * rinv, cj = eG * Ai * rinv;
    float rad = P.eps_patch * dG * Ai * Aj;
    // dV/dr_vec = -[ rad*u + ci*(S_i - siu u) - cj*(S_j - sju u) ] ; F_j = -dV/dr_vec
    fx = rad * ux + ci * (Six - siu * ux) - cj * (Sjx - sju * ux);
    fy = rad * uy + ci * (Siy - siu * uy) - cj * (Sjy - sju * uy);
    fz = rad * uz + ci * (Siz - siu * uz) - cj * (Sjz - sju * uz);
    // tau_i = eps_p G A_j (S_i x u)
    float ti = eG * Aj;
    tix = ti * (Siy * uz - Siz * uy); tiy = ti * (Siz * ux - Six * uz); tiz = ti * (Six * uy - Siy * ux);
    if (NEED_TJ) {   // tau_j = eps_p G A_i (S_j x (-u))
        float tj = -eG * Ai;
        tjx = tj * (Sjy * uz - Sjz * uy); tjy = tj * (Sjz * ux - Sjx * uz); tjz = tj * (Sjx * uy - Sjy * ux);
    }
    if (d2 < P.core_rc2) {   // WCA core (force continuous at its cut: plain fp32 test)
        float inv = rinv * rinv;
        float s2 = P.sig2 * inv, s6 = s2 * s2 * s2;
        float g = inv * s6 * fmaf(P.c48, s6, -P.c24);
        V += fmaf(s6, fmaf(P.c4, s6, -P.c4), -P.core_vshift);
        fx = fmaf(g, dx, fx); fy = fmaf(g, dy, fy); fz = fmaf(g, dz, fz);
    }
}

// the rigid-body pair function a kernel instance is compiled for: PP = the paper's own model (S:8(f2)), else config 4's
__host__ __device__ constexpr bool md_is_rigid(int kind) { return kind == MD_POT_PATCHY || kind == MD_POT_PATCHY_PP; }
template <bool NEED_TJ, bool PP>
__device__ __forceinline__ void rigid_pair(const DevParams& P, float dx, float dy, float dz, float d2, const Rot& Ri, float4 qj,
                                           float& fx, float& fy, float& fz, float& V,
                                           float& tix, float& tiy, float& tiz, float& tjx, float& tjy, float& tjz) {
    if (PP) patchy_pp_pair<NEED_TJ>(P, dx, dy, dz, d2, Ri, qj, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
    else if (P.n_patches == 4) patchy_pair<NEED_TJ, 4>(P, dx, dy, dz, d2, Ri, qj, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
    else patchy_pair<NEED_TJ, 0>(P, dx, dy, dz, d2, Ri, qj, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
}

// O3 FENE (B:9): U = -1/2 K R0^2 ln(1 - d2/R0^2); force on j = -K d / (1 - d2/R0^2)
__device__ __forceinline__ bool fene_pair(const DevParams& P, float d2, float& g, float& V) {
    float q = 1.0f - d2 * P.fene_invR02;
    if (!(q > 0.0f)) { g = 0.f; V = 0.f; return false; }
    g = -P.fene_K / q;
    V = -0.5f * P.fene_K * P.fene_R02 * __logf(q);
    return true;
}

