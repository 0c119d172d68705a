// md_integrate.cu -- velocity-Verlet NVE in fp32 state (S:A10, S:O6; rigid bodies S:O7), the skin
// criterion (S:A5, S:Q4) and the energy reduction (S:A9).
#include <stdio.h>
#include "md_internal.cuh"

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// first half: v += dt/2 F/m ; [L += dt/2 tau ; q <- dq (x) q] ; x += dt v ; skin check.
// PRE: the closing half kick of the previous step is applied first, in this kernel (same two roundings as k_kick
// followed by this kernel: inside a multi-step graph the separate k_kick launch and its pass over vel/force are saved).
template <bool RIGID, bool PRE>
__global__ void __launch_bounds__(256) k_kick_drift(DevParams P, DevBuffers B, float dt, float4* pos, float4* __restrict__ vel,
                                                    const float4* __restrict__ force, float4* __restrict__ quat,
                                                    float4* __restrict__ angmom, const float4* __restrict__ torque,
                                                    float4* pos_out) {      // == pos, or the other position array (fused steps)
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < P.N) {
        // ghosts of a space decomposition (md_set_active) are moved by the halo refresh only; their skin check still runs
        const bool ghost = P.n_active < P.N && B.ids[i] >= P.n_active;
        const float hk = ghost ? 0.0f : 0.5f * dt * P.inv_mass;
        if (ghost) dt = 0.0f;
        float4 v = vel[i], f = force[i], x = pos[i];
        if (PRE) { v.x = fmaf(hk, f.x, v.x); v.y = fmaf(hk, f.y, v.y); v.z = fmaf(hk, f.z, v.z); }
        v.x = fmaf(hk, f.x, v.x); v.y = fmaf(hk, f.y, v.y); v.z = fmaf(hk, f.z, v.z);
        x.x = fmaf(dt, v.x, x.x); x.y = fmaf(dt, v.y, x.y); x.z = fmaf(dt, v.z, x.z);
        vel[i] = v;
        pos_out[i] = x;
        if (RIGID && !ghost) {
            float4 L = angmom[i], t = torque[i], q = quat[i];
            const float hd = 0.5f * dt;
            if (PRE) { L.x = fmaf(hd, t.x, L.x); L.y = fmaf(hd, t.y, L.y); L.z = fmaf(hd, t.z, L.z); }
            L.x = fmaf(hd, t.x, L.x); L.y = fmaf(hd, t.y, L.y); L.z = fmaf(hd, t.z, L.z);
            angmom[i] = L;
            float wx = L.x * P.inv_inertia, wy = L.y * P.inv_inertia, wz = L.z * P.inv_inertia;
            float wn = sqrtf(wx * wx + wy * wy + wz * wz);
            if (wn > 0.0f) {   // exact free rotation of a spherical top about the space-frame axis omega (S:O7)
                float h = 0.5f * wn * dt, sn, c;
                sincosf(h, &sn, &c);
                sn /= wn;
                float a0 = c, a1 = sn * wx, a2 = sn * wy, a3 = sn * wz;
                float q0 = q.x, q1 = q.y, q2 = q.z, q3 = q.w;   // (w,x,y,z)
                float r0 = a0 * q0 - a1 * q1 - a2 * q2 - a3 * q3;
                float r1 = a0 * q1 + a1 * q0 + a2 * q3 - a3 * q2;
                float r2 = a0 * q2 - a1 * q3 + a2 * q0 + a3 * q1;
                float r3 = a0 * q3 + a1 * q2 - a2 * q1 + a3 * q0;
                float nrm = rsqrtf(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3);
                quat[i] = make_float4(r0 * nrm, r1 * nrm, r2 * nrm, r3 * nrm);
            }
        }
        float4 r = B.pos_ref[i];
        float dx = x.x - r.x, dy = x.y - r.y, dz = x.z - r.z;
        moved = (dx * dx + dy * dy + dz * dz) > P.half_skin2;   // S:Q4 strict '>'
    }
    if (__any_sync(0xffffffffu, moved) && (threadIdx.x & 31) == 0) B.ctrl->rebuild = 1;
}

// second half: v += dt/2 F/m ; L += dt/2 tau
template <bool RIGID>
__global__ void __launch_bounds__(256) k_kick(DevParams P, DevBuffers B, float dt, float4* __restrict__ vel, const float4* __restrict__ force,
                                              float4* __restrict__ angmom, const float4* __restrict__ torque) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    if (P.n_active < P.N && B.ids[i] >= P.n_active) return;   // ghost (md_set_active)
    const float hk = 0.5f * dt * P.inv_mass;
    float4 v = vel[i], f = force[i];
    v.x = fmaf(hk, f.x, v.x); v.y = fmaf(hk, f.y, v.y); v.z = fmaf(hk, f.z, v.z);
    vel[i] = v;
    if (RIGID) {
        float4 L = angmom[i], t = torque[i];
        const float hd = 0.5f * dt;
        L.x = fmaf(hd, t.x, L.x); L.y = fmaf(hd, t.y, L.y); L.z = fmaf(hd, t.z, L.z);
        angmom[i] = L;
    }
}

// ------------------------------------------------------------------------------------------------
// Mixed precision (S:8(f3)): the same two kernels on the fp64 copies of the state; forces and torques stay
// fp32, the fp32 arrays are rewritten (round to nearest) for the force kernels, the skin check and the caller.
// ------------------------------------------------------------------------------------------------
template <bool RIGID, bool PRE>
__global__ void __launch_bounds__(256) k_kick_drift_mixed(DevParams P, DevBuffers B, double dt, float4* pos, float4* vel,
                                                          const float4* __restrict__ force, float4* quat, float4* angmom,
                                                          const float4* __restrict__ torque) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < P.N) {
        double2* pxy = reinterpret_cast<double2*>(B.shadow[0]); double2* pz = reinterpret_cast<double2*>(B.shadow[1]);
        double2* vxy = reinterpret_cast<double2*>(B.shadow[2]); double2* vz = reinterpret_cast<double2*>(B.shadow[3]);
        const double hk = 0.5 * dt / (double)P.mass;
        const float4 f = force[i];
        double2 xa = pxy[i], xb = pz[i], va = vxy[i], vb = vz[i];
        if (PRE) { va.x = fma(hk, (double)f.x, va.x); va.y = fma(hk, (double)f.y, va.y); vb.x = fma(hk, (double)f.z, vb.x); }
        va.x = fma(hk, (double)f.x, va.x); va.y = fma(hk, (double)f.y, va.y); vb.x = fma(hk, (double)f.z, vb.x);
        xa.x = fma(dt, va.x, xa.x); xa.y = fma(dt, va.y, xa.y); xb.x = fma(dt, vb.x, xb.x);
        pxy[i] = xa; pz[i] = xb; vxy[i] = va; vz[i] = vb;
        float4 x = pos[i], v = vel[i];
        x.x = (float)xa.x; x.y = (float)xa.y; x.z = (float)xb.x;
        v.x = (float)va.x; v.y = (float)va.y; v.z = (float)vb.x;
        pos[i] = x; vel[i] = v;
        if (RIGID) {
            double2* lxy = reinterpret_cast<double2*>(B.shadow[4]); double2* lz = reinterpret_cast<double2*>(B.shadow[5]);
            double2* qa = reinterpret_cast<double2*>(B.shadow[6]); double2* qb = reinterpret_cast<double2*>(B.shadow[7]);
            const float4 t = torque[i];
            const double hd = 0.5 * dt;
            double2 La = lxy[i], Lb = lz[i];
            if (PRE) { La.x = fma(hd, (double)t.x, La.x); La.y = fma(hd, (double)t.y, La.y); Lb.x = fma(hd, (double)t.z, Lb.x); }
            La.x = fma(hd, (double)t.x, La.x); La.y = fma(hd, (double)t.y, La.y); Lb.x = fma(hd, (double)t.z, Lb.x);
            lxy[i] = La; lz[i] = Lb;
            float4 L = angmom[i];
            L.x = (float)La.x; L.y = (float)La.y; L.z = (float)Lb.x;
            angmom[i] = L;
            const double inv_I = (double)P.inv_inertia;
            const double wx = La.x * inv_I, wy = La.y * inv_I, wz = Lb.x * inv_I;
            const double wn = sqrt(wx * wx + wy * wy + wz * wz);
            if (wn > 0.0) {   // S:O7, as k_kick_drift
                double sn, c;
                sincos(0.5 * wn * dt, &sn, &c);
                sn /= wn;
                const double a0 = c, a1 = sn * wx, a2 = sn * wy, a3 = sn * wz;
                const double2 q01 = qa[i], q23 = qb[i];
                const double q0 = q01.x, q1 = q01.y, q2 = q23.x, q3 = q23.y;
                double r0 = a0 * q0 - a1 * q1 - a2 * q2 - a3 * q3;
                double r1 = a0 * q1 + a1 * q0 + a2 * q3 - a3 * q2;
                double r2 = a0 * q2 - a1 * q3 + a2 * q0 + a3 * q1;
                double r3 = a0 * q3 + a1 * q2 - a2 * q1 + a3 * q0;
                const double nrm = 1.0 / sqrt(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3);
                r0 *= nrm; r1 *= nrm; r2 *= nrm; r3 *= nrm;
                qa[i] = make_double2(r0, r1); qb[i] = make_double2(r2, r3);
                quat[i] = make_float4((float)r0, (float)r1, (float)r2, (float)r3);
            }
        }
        const float4 r = B.pos_ref[i];
        const float dx = x.x - r.x, dy = x.y - r.y, dz = x.z - r.z;
        moved = (dx * dx + dy * dy + dz * dz) > P.half_skin2;   // S:Q4, on the fp32 positions the lists were built from
    }
    if (__any_sync(0xffffffffu, moved) && (threadIdx.x & 31) == 0) B.ctrl->rebuild = 1;
}

template <bool RIGID>
__global__ void __launch_bounds__(256) k_kick_mixed(DevParams P, DevBuffers B, double dt, float4* vel, const float4* __restrict__ force,
                                                    float4* angmom, const float4* __restrict__ torque) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    double2* vxy = reinterpret_cast<double2*>(B.shadow[2]); double2* vz = reinterpret_cast<double2*>(B.shadow[3]);
    const double hk = 0.5 * dt / (double)P.mass;
    const float4 f = force[i];
    double2 va = vxy[i], vb = vz[i];
    va.x = fma(hk, (double)f.x, va.x); va.y = fma(hk, (double)f.y, va.y); vb.x = fma(hk, (double)f.z, vb.x);
    vxy[i] = va; vz[i] = vb;
    float4 v = vel[i];
    v.x = (float)va.x; v.y = (float)va.y; v.z = (float)vb.x;
    vel[i] = v;
    if (RIGID) {
        double2* lxy = reinterpret_cast<double2*>(B.shadow[4]); double2* lz = reinterpret_cast<double2*>(B.shadow[5]);
        const float4 t = torque[i];
        const double hd = 0.5 * dt;
        double2 La = lxy[i], Lb = lz[i];
        La.x = fma(hd, (double)t.x, La.x); La.y = fma(hd, (double)t.y, La.y); Lb.x = fma(hd, (double)t.z, Lb.x);
        lxy[i] = La; lz[i] = Lb;
        float4 L = angmom[i];
        L.x = (float)La.x; L.y = (float)La.y; L.z = (float)Lb.x;
        angmom[i] = L;
    }
}

// fp64 copies <- the bound fp32 arrays (exact)
__global__ void __launch_bounds__(256) k_shadow_init(DevParams P, DevBuffers B, const float4* __restrict__ pos, const float4* __restrict__ vel,
                                                     const float4* __restrict__ quat, const float4* __restrict__ angmom) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const float4 x = pos[i], v = vel[i];
    reinterpret_cast<double2*>(B.shadow[0])[i] = make_double2((double)x.x, (double)x.y);
    reinterpret_cast<double2*>(B.shadow[1])[i] = make_double2((double)x.z, 0.0);
    reinterpret_cast<double2*>(B.shadow[2])[i] = make_double2((double)v.x, (double)v.y);
    reinterpret_cast<double2*>(B.shadow[3])[i] = make_double2((double)v.z, 0.0);
    if (quat) {
        const float4 q = quat[i], L = angmom[i];
        reinterpret_cast<double2*>(B.shadow[4])[i] = make_double2((double)L.x, (double)L.y);
        reinterpret_cast<double2*>(B.shadow[5])[i] = make_double2((double)L.z, 0.0);
        reinterpret_cast<double2*>(B.shadow[6])[i] = make_double2((double)q.x, (double)q.y);
        reinterpret_cast<double2*>(B.shadow[7])[i] = make_double2((double)q.z, (double)q.w);
    }
}

void md_launch_shadow_init(md_system* s) {
    k_shadow_init<<<cdiv(s->P.N, 256), 256, 0, s->stream>>>(s->P, s->B, s->pos, s->vel, s->rigid ? s->quat : nullptr, s->rigid ? s->angmom : nullptr);
    s->launches += 1;
}

// drives the IF node of the step graph: run the rebuild body iff the skin criterion tripped (S:A5)
__global__ void k_set_cond(cudaGraphConditionalHandle h, DevBuffers B) { cudaGraphSetConditional(h, B.ctrl->rebuild != 0 ? 1u : 0u); }

void md_launch_set_cond(md_system* s, unsigned long long cond_handle) {
    k_set_cond<<<1, 1, 0, s->stream>>>((cudaGraphConditionalHandle)cond_handle, s->B);
    s->launches += 1;
}

void md_launch_kick_drift_to(md_system* s, float dt, float4* pos_out) {
    k_kick_drift<false, false><<<cdiv(s->P.N, 256), 256, 0, s->stream>>>(s->P, s->B, dt, s->pos, s->vel, s->force, nullptr, nullptr, nullptr, pos_out);
    s->launches += 1;
}

void md_launch_kick_drift(md_system* s, float dt, bool pre) {
    int nb = cdiv(s->P.N, 256);
    if (s->precision == MD_PREC_MIXED) {
        const double d = s->dt_d;
        if (s->rigid) {
            if (pre) k_kick_drift_mixed<true, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, d, s->pos, s->vel, s->force, s->quat, s->angmom, s->torque);
            else k_kick_drift_mixed<true, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, d, s->pos, s->vel, s->force, s->quat, s->angmom, s->torque);
        } else {
            if (pre) k_kick_drift_mixed<false, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, d, s->pos, s->vel, s->force, nullptr, nullptr, nullptr);
            else k_kick_drift_mixed<false, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, d, s->pos, s->vel, s->force, nullptr, nullptr, nullptr);
        }
        s->launches += 1;
        return;
    }
    if (s->rigid) {
        if (pre) k_kick_drift<true, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->pos, s->vel, s->force, s->quat, s->angmom, s->torque, s->pos);
        else k_kick_drift<true, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->pos, s->vel, s->force, s->quat, s->angmom, s->torque, s->pos);
    } else {
        if (pre) k_kick_drift<false, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->pos, s->vel, s->force, nullptr, nullptr, nullptr, s->pos);
        else k_kick_drift<false, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->pos, s->vel, s->force, nullptr, nullptr, nullptr, s->pos);
    }
    s->launches += 1;
}

void md_launch_kick(md_system* s, float dt) {
    int nb = cdiv(s->P.N, 256);
    if (s->precision == MD_PREC_MIXED) {
        if (s->rigid) k_kick_mixed<true><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->dt_d, s->vel, s->force, s->angmom, s->torque);
        else k_kick_mixed<false><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->dt_d, s->vel, s->force, nullptr, nullptr);
        s->launches += 1;
        return;
    }
    if (s->rigid) k_kick<true><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->vel, s->force, s->angmom, s->torque);
    else k_kick<false><<<nb, 256, 0, s->stream>>>(s->P, s->B, dt, s->vel, s->force, nullptr, nullptr);
    s->launches += 1;
}

// ------------------------------------------------------------------------------------------------
// S:8(f3), "the thermostat described in Ref. 27" -- reading DESIGN.md QT: Andersen-type velocity refresh.
// One thread per slot; the random stream belongs to the ORIGINAL id (B.ids), so the result does not depend on the
// storage order.  Philox4x32-10, key = seed words, counter = (id, application index, stream, block): block 0 word 0
// decides by an integer comparison, block 1 gives three Gaussians by Box-Muller in fp64 (p N particles every n_newt
// steps: fp64 here costs nothing, and the draw is then exact to the fp32 rounding of the stored velocity).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned int h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x;
        const unsigned int h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
        c = make_uint4(h1 ^ c.y ^ k.x, l1, h0 ^ c.w ^ k.y, l0);
        k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ bool thermostat_decide(unsigned int id, unsigned int call, unsigned int stream, uint2 key, unsigned long long thr) {
    return (unsigned long long)philox4x32_10(make_uint4(id, call, stream, 0u), key).x < thr;
}

__device__ __forceinline__ void thermostat_gauss(unsigned int id, unsigned int call, unsigned int stream, uint2 key, double g[3]) {
    const uint4 w = philox4x32_10(make_uint4(id, call, stream, 1u), key);
    const double sc = 1.0 / 4294967296.0;
    const double u0 = ((double)w.x + 0.5) * sc, u1 = ((double)w.y + 0.5) * sc;
    const double u2 = ((double)w.z + 0.5) * sc, u3 = ((double)w.w + 0.5) * sc;
    const double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
    double sn, cs, sn2, cs2;
    sincospi(2.0 * u1, &sn, &cs);
    sincospi(2.0 * u3, &sn2, &cs2);
    g[0] = r0 * cs; g[1] = r0 * sn; g[2] = r1 * cs2;
}

// Two phases per block: every thread takes the integer decisions of its slot (Philox block 0) and appends the
// refreshed (slot, stream) to a shared-memory list; then the list is worked off with full warps, so the fp64
// Box-Muller runs on ~p x 256 lanes instead of dragging every warp through it for its few refreshed lanes.
#define THERMO_ITEMS 4     // slots per thread: 1024 decisions per block amortise the two barriers and fill the second phase
template <bool RIGID, bool MIXED>
__global__ void __launch_bounds__(256) k_thermostat(DevParams P, DevBuffers B, float4* __restrict__ vel, float4* __restrict__ angmom,
                                                    double sv, double sl, unsigned long long thr_t, unsigned long long thr_r,
                                                    uint2 key, unsigned int call) {
    __shared__ unsigned int todo[2 * 256 * THERMO_ITEMS];      // slot | stream << 31
    __shared__ unsigned int todo_id[2 * 256 * THERMO_ITEMS];   // original id of that slot
    __shared__ int ntodo;
    if (threadIdx.x == 0) ntodo = 0;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < THERMO_ITEMS; ++k) {
        const int i = (blockIdx.x * THERMO_ITEMS + k) * 256 + threadIdx.x;
        if (i < P.N) {
            const unsigned int id = (unsigned int)B.ids[i];
            if (thermostat_decide(id, call, 0u, key, thr_t)) {
                const int q = atomicAdd(&ntodo, 1);
                todo[q] = (unsigned int)i; todo_id[q] = id;
            }
            if (RIGID && thermostat_decide(id, call, 1u, key, thr_r)) {
                const int q = atomicAdd(&ntodo, 1);
                todo[q] = (unsigned int)i | 0x80000000u; todo_id[q] = id;
            }
        }
    }
    __syncthreads();
    const int n = ntodo;
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const unsigned int e = todo[k], stream = e >> 31;
        const int slot = (int)(e & 0x7fffffffu);
        float4* arr = stream ? angmom : vel;
        float4 v = arr[slot];                  // keeps the w component; requested before the fp64 chain
        double g[3];
        thermostat_gauss(todo_id[k], call, stream, key, g);
        const double sc = stream ? sl : sv;
        const double a = sc * g[0], b = sc * g[1], c = sc * g[2];
        v.x = (float)a; v.y = (float)b; v.z = (float)c;
        arr[slot] = v;
        if (MIXED) {
            reinterpret_cast<double2*>(B.shadow[stream ? 4 : 2])[slot] = make_double2(a, b);
            reinterpret_cast<double2*>(B.shadow[stream ? 5 : 3])[slot] = make_double2(c, 0.0);
        }
    }
}

static unsigned long long thermostat_threshold(double p) {
    const double t = floor(p * 4294967296.0);
    return t <= 0.0 ? 0ull : (t >= 4294967296.0 ? 4294967296ull : (unsigned long long)t);
}

void md_launch_thermostat(md_system* s, double T, double p_t, double p_r, unsigned long long seed, unsigned int call) {
    const int nb = cdiv(s->P.N, 256 * THERMO_ITEMS);
    const double sv = sqrt(T / (double)s->pot.mass), sl = s->rigid ? sqrt(T * (double)s->pot.inertia) : 0.0;
    const unsigned long long tt = thermostat_threshold(p_t), tr = thermostat_threshold(p_r);
    const uint2 key = make_uint2((unsigned int)(seed & 0xffffffffull), (unsigned int)(seed >> 32));
    const bool mixed = s->precision == MD_PREC_MIXED;
    if (s->rigid) {
        if (mixed) k_thermostat<true, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->vel, s->angmom, sv, sl, tt, tr, key, call);
        else k_thermostat<true, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->vel, s->angmom, sv, sl, tt, tr, key, call);
    } else {
        if (mixed) k_thermostat<false, true><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->vel, nullptr, sv, sl, tt, tr, key, call);
        else k_thermostat<false, false><<<nb, 256, 0, s->stream>>>(s->P, s->B, s->vel, nullptr, sv, sl, tt, tr, key, call);
    }
    s->launches += 1;
}

// ------------------------------------------------------------------------------------------------
// S:A9 energies: fp32 per-particle terms accumulated in fp64, two deterministic stages
// ------------------------------------------------------------------------------------------------
#define E_THREADS 256
#define E_BLOCKS 2048   // capacity of the partial-sum table (md_api.cu carve: e_part); the launch uses 8 blocks per SM

__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
    }
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(E_THREADS) k_energy_partial(DevParams P, DevBuffers B, const float4* __restrict__ vel,
                                                             const float4* __restrict__ force, const float4* __restrict__ angmom) {
    __shared__ double sh[32];
    double u = 0.0, kt = 0.0, kr = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        if (P.n_active < P.N && B.ids[i] >= P.n_active) continue;   // ghosts belong to another rank's sums (md_set_active)
        u += (double)force[i].w;
        float4 v = vel[i];
        kt += (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z;
        if (angmom) {
            float4 L = angmom[i];
            kr += (double)L.x * L.x + (double)L.y * L.y + (double)L.z * L.z;
        }
    }
    u = block_sum(u, sh); kt = block_sum(kt, sh); kr = block_sum(kr, sh);
    if (threadIdx.x == 0) {
        B.e_part[3 * blockIdx.x + 0] = u;
        B.e_part[3 * blockIdx.x + 1] = kt;
        B.e_part[3 * blockIdx.x + 2] = kr;
    }
}

__global__ void __launch_bounds__(E_THREADS) k_energy_final(DevParams P, DevBuffers B, int nblocks) {
    __shared__ double sh[32];
    double u = 0.0, kt = 0.0, kr = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
        u += B.e_part[3 * b + 0]; kt += B.e_part[3 * b + 1]; kr += B.e_part[3 * b + 2];
    }
    u = block_sum(u, sh); kt = block_sum(kt, sh); kr = block_sum(kr, sh);
    if (threadIdx.x == 0) {
        B.e_out[0] = u;
        B.e_out[1] = 0.5 * (double)P.mass * kt;
        B.e_out[2] = 0.5 * (double)P.inv_inertia * kr;
    }
}

void md_launch_energy(md_system* s) {
    int nb = cdiv(s->P.N, E_THREADS);
    if (nb > s->sm_count * 8) nb = s->sm_count * 8;
    if (nb > E_BLOCKS) nb = E_BLOCKS;
    k_energy_partial<<<nb, E_THREADS, 0, s->stream>>>(s->P, s->B, s->vel, s->force, s->rigid ? s->angmom : nullptr);
    k_energy_final<<<1, E_THREADS, 0, s->stream>>>(s->P, s->B, nb);
    s->launches += 2;
}
