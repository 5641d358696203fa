// dem_kernels.cuh -- the CUDA kernels of libdem_b200 (sm_100a).  Host orchestration is in dem_lib.cu.
//
//   a3-a7 pair-feature kernel           k_pair          (FP32-ALU bound; dem_math.cuh holds the arithmetic)
//   a8  per-particle reduction          k_finish        (one thread per particle, no atomics; fused with the integrator)
// The neighbour-list kernels (a2) are in dem_list.cuh, the integrator (a9) in dem_integrate.cuh, the packed FP32 search
// kernels in dem_fast.cuh.
#pragma once
#include <cuda_runtime.h>

#include "dem_math.cuh"
#include "dem_rigid.cuh"

namespace dem {

// ---- loads --------------------------------------------------------------------------------------------------------
__device__ __forceinline__ d4 load4d(const float* p, int i) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(p) + i);
    d4 r;
    r.x = v.x; r.y = v.y; r.z = v.z; r.w = v.w;
    return r;
}
__device__ __forceinline__ d4 load4d(const double* p, int i) {
    const double2 a = __ldg(reinterpret_cast<const double2*>(p) + 2 * (size_t)i);
    const double2 b = __ldg(reinterpret_cast<const double2*>(p) + 2 * (size_t)i + 1);
    d4 r;
    r.x = a.x; r.y = a.y; r.z = b.x; r.w = b.y;
    return r;
}

// Minimum image with the operation order both sides of the bit-exact neighbour test use (R13):
// d = x_j - x_i; d -= L * rint(d / L), each operation rounded separately (no FMA contraction).
// The quotient is formed as da * (1/L), which lies within 2 ulp of the correctly rounded da / L: unless it is that
// close to a half-integer (where the division is carried out) both round to the same integer, so the result is the
// one the definition gives, bit for bit, at the cost of a multiplication instead of an FP64 division.
__device__ __forceinline__ double min_image_1(double xi, double xj, double L, double invL) {
    const double da = __dsub_rn(xj, xi);
    const double t = __dmul_rn(da, invL);
    double k = rint(t);
    if (fabs(fabs(t - k) - 0.5) < 1e-9 * (1.0 + fabs(t))) k = rint(__ddiv_rn(da, L));
    return __dsub_rn(da, __dmul_rn(L, k));
}
__device__ __forceinline__ double norm2_fma(double dx, double dy, double dz) {
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}

// ---- a3-a7: the pair-feature kernel ---------------------------------------------------------------------------------
template <typename real, typename PosT, int DIM>
__global__ void __launch_bounds__(128) k_pair(const PairArgs<real> a) {
    typedef typename vec4<real>::type real4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    real4* sm = reinterpret_cast<real4*>(smem_raw);
    // stage the shape-feature tables of the class (a1) into shared memory
    const bool same = a.sa.off == a.sb.off;
    for (int k = threadIdx.x; k < a.sa.len; k += blockDim.x) sm[k] = a.table[a.sa.off + k];
    if (!same)
        for (int k = threadIdx.x; k < a.sb.len; k += blockDim.x) sm[a.sa.len + k] = a.table[a.sb.off + k];
    __syncthreads();
    ShapeView<real> A, B;
    A.nv = a.sa.nv; A.ne = a.sa.ne; A.nf = a.sa.nf;
    A.V = sm; A.E = A.V + A.nv; A.F = A.E + 2 * A.ne; A.FE = A.F + 4 * A.nf; A.OE = A.FE + 2 * a.sa.nfe;
    B.nv = a.sb.nv; B.ne = a.sb.ne; B.nf = a.sb.nf;
    B.V = same ? sm : sm + a.sa.len; B.E = B.V + B.nv; B.F = B.E + 2 * B.ne; B.FE = B.F + 4 * B.nf;
    B.OE = B.FE + 2 * a.sb.nfe;

    const int np_pad = (a.npairs + 31) & ~31;  // slices are warp-uniform
    const long long n_items = (long long)np_pad * a.slices;
    unsigned c_eval = 0, c_act = 0, c_deg = 0, c_par = 0;
    for (long long item = (long long)blockIdx.x * blockDim.x + threadIdx.x; item < n_items;
         item += (long long)gridDim.x * blockDim.x) {
        const int slice = (int)(item / np_pad), p = (int)(item - (long long)slice * np_pad);
        if (p >= a.npairs) continue;
        const int2 ij = a.pairs[p];
        const d4 xi = load4d(static_cast<const PosT*>(a.pos), ij.x), xj = load4d(static_cast<const PosT*>(a.pos), ij.y);
        double d[3];
        d[0] = min_image_1(xi.x, xj.x, a.box.L[0], a.box.invL[0]);
        d[1] = min_image_1(xi.y, xj.y, a.box.L[1], a.box.invL[1]);
        d[2] = DIM == 3 ? min_image_1(xi.z, xj.z, a.box.L[2], a.box.invL[2]) : 0.0;
        real out[10];
#pragma unroll
        for (int k = 0; k < 10; ++k) out[k] = real(0);
        unsigned nact = 0u;
        if (d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < a.reach2) {
            const d4 qi = load4d(static_cast<const PosT*>(a.quat), ij.x), qj = load4d(static_cast<const PosT*>(a.quat), ij.y);
            const double qa[4] = {qi.x, qi.y, qi.z, qi.w}, qb[4] = {qj.x, qj.y, qj.z, qj.w};
            const int ob = (int)((long long)slice * a.n_outer / a.slices);
            const int oe = (int)((long long)(slice + 1) * a.n_outer / a.slices);
            unsigned cnt[3];
            pair_lab<real, DIM>(A, B, qa, qb, d, a.pc, ob, oe, out, cnt);
            c_eval += slice == 0;
            c_act += cnt[0];
            c_deg += cnt[1];
            c_par += cnt[2];
            nact = cnt[0];
        }
        // result record (DEM_REC real4 each): (F_i, U_ij) (tau_i, d.x) (d.y, d.z, 0, 0); the reduction derives the other
        // side: F_j = -F_i, tau_j = -tau_i + d x F_i.  Written only when a term is inside the cutoff; the flag tells the
        // reduction whether there is a record to read.
        const size_t ri = (size_t)p * a.slices + slice;
        a.rflag[ri] = nact ? 1 : 0;
        if (nact) {
            real4* rec = a.rec + DEM_REC * ri;
            real4 r0, r1, r2;
            r0.x = out[0]; r0.y = out[1]; r0.z = out[2]; r0.w = out[9];
            r1.x = out[3]; r1.y = out[4]; r1.z = out[5]; r1.w = (real)d[0];
            r2.x = (real)d[1]; r2.y = (real)d[2]; r2.z = r2.w = real(0);
            rec[0] = r0; rec[1] = r1; rec[2] = r2;
        }
    }
    // counters: one atomic per warp per counter, after the hot loop
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        c_eval += __shfl_xor_sync(0xffffffffu, c_eval, o);
        c_act += __shfl_xor_sync(0xffffffffu, c_act, o);
        c_deg += __shfl_xor_sync(0xffffffffu, c_deg, o);
        c_par += __shfl_xor_sync(0xffffffffu, c_par, o);
    }
    if ((threadIdx.x & 31) == 0 && a.counters) {  // null inside dem_step: counters belong to dem_compute
        if (c_eval) atomicAdd(a.counters + 0, (unsigned long long)c_eval);
        if (c_act) atomicAdd(a.counters + 1, (unsigned long long)c_act);
        if (c_deg) atomicAdd(a.counters + 2, (unsigned long long)c_deg);
        if (c_par) atomicAdd(a.counters + 3, (unsigned long long)c_par);
    }
}

// ---- a8 (+ a9): per-particle reduction, fused with the integrator ------------------------------------------------------
// a particle's total is the sum over its neighbours.  One thread per particle walks its neighbour slots
// (slot[k][i], neighbour-major so that a warp's loads coalesce: 2 x pair index + which side of the pair the particle is;
// the pair's class follows from the class-major pair index), looks up each pair's record flag and reads the 48-byte
// record only where a term was inside the cutoff.  The loads of a batch of four neighbours are issued before any is
// used.  The summation order is fixed (no atomics), so results are bit-reproducible from run to run.
// Inside dem_step the same thread goes on with the integrator (FinArgs: second half kick; in mode 2 also the first
// half kick of the next step, the drift, the free rotation and the skin test), which saves the passes over F, tau, v
// and L that separate kernels would need.  Forces and torques are stored only in modes 0 and 1 (mode 2 consumes them
// in registers; the step that ends a dem_step call runs in mode 1).
#define DEM_FIN_W 8
template <typename real, int MODE>
__global__ void __launch_bounds__(256) k_finish(int N, int stride, const int* __restrict__ slot,
                                                const int* __restrict__ sid, ClassTable ct, int nclass,
                                                const typename vec4<real>::type* __restrict__ rec,
                                                const unsigned char* __restrict__ rflag,
                                                typename vec4<real>::type* __restrict__ force,
                                                typename vec4<real>::type* __restrict__ torque, real* __restrict__ virial,
                                                FinArgs fa) {
    typedef typename vec4<real>::type real4;
    // fa.lanes lanes share a particle (1 for large systems; small ones are bound by the latency of the serial walk over
    // a particle's slots, so several lanes split it and combine with shuffles: still a fixed order for a given N)
    const int lpp = fa.lanes, gid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = gid / lpp, sub = gid - i * lpp;
    // The kernel is a chain of dependent loads (stale flag -> slots -> record flags -> state): ask the L2 for everything
    // whose address is known now, so that the chain runs on L2 hits
    if (i < N) {
#pragma unroll
        for (int u = 0; u < DEM_FIN_W; ++u)
            if (DEM_FIN_W * sub + u < stride)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(slot + (size_t)(DEM_FIN_W * sub + u) * N + i));
        if (MODE >= 1 && sub == 0) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.vel + i));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.ang + i));
            if (MODE == 2) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.pos + i));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.quat + i));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.pos_build + i));
            }
        }
    }
    if (MODE != 0) {
        if (fa.bail && *fa.bail) {               // the list went stale before this step: change nothing, and pass
            if (gid == 0 && fa.raise) *fa.raise = 1;  // the word on (the next evaluation looks at the other flag)
            return;
        }
        if (gid == 0 && fa.done) *fa.done += 1;  // nothing in this kernel reads it
    }
    const bool live = i < N, lead = live && sub == 0;
    real F[3] = {0, 0, 0}, T[3] = {0, 0, 0}, U = 0, W[6] = {0, 0, 0, 0, 0, 0};
    // A particle's slots are walked DEM_FIN_W at a time: the slot loads of a batch are in flight together, then its flag
    // loads.  Rows end with -1 (k_slot_back pads them), so the walk does not wait for the particle's neighbour count.
    for (int k0 = DEM_FIN_W * sub; live && k0 < stride; k0 += DEM_FIN_W * lpp) {
        int sl[DEM_FIN_W];
        int ri[DEM_FIN_W];   // (record indices fit an int: checked at the build)
        int S[DEM_FIN_W];
        unsigned any[DEM_FIN_W];
#pragma unroll
        for (int u = 0; u < DEM_FIN_W; ++u) sl[u] = k0 + u < stride ? slot[(size_t)(k0 + u) * N + i] : -1;
        if (sl[0] < 0) break;
#pragma unroll
        for (int u = 0; u < DEM_FIN_W; ++u) {
            any[u] = 0u;
            S[u] = 0;
            ri[u] = 0;
            if (sl[u] >= 0) {
                const int p = sl[u] >> 1;
                int c = 0;
                while (c + 1 < nclass && p >= ct.pair_base[c + 1]) ++c;
                DEM_ASSERT(p < ct.pair_base[nclass] && p >= ct.pair_base[c]);
                S[u] = ct.slices[c];
                ri[u] = ct.rec_base[c] + (p - ct.pair_base[c]) * S[u];
                // bit s: slice s of the pair has a record (more than 32 slices: every flag is looked at below)
                for (int s = 0; s < S[u] && s < 32; ++s) any[u] |= (unsigned)(rflag[ri[u] + s] != 0) << s;
                if (S[u] > 32) any[u] |= 0x80000000u;
            }
        }
#pragma unroll
        for (int u = 0; u < DEM_FIN_W; ++u) {
            if (!any[u]) continue;  // this pair contributes nothing: no record was written
            const int side = sl[u] & 1;
            for (int s = 0; s < S[u]; ++s) {
                if (S[u] <= 32 ? !((any[u] >> s) & 1u) : !rflag[ri[u] + s]) continue;
                const real4* r = rec + DEM_REC * (size_t)(ri[u] + s);
                const real4 r0 = r[0], r1 = r[1], r2 = r[2];
                const real dx = r1.w, dy = r2.x, dz = r2.y;
                if (side) {  // this particle is the pair's second one: F_j = -F_i, tau_j = -tau_i + d x F_i
                    F[0] -= r0.x; F[1] -= r0.y; F[2] -= r0.z;
                    T[0] += (dy * r0.z - dz * r0.y) - r1.x;
                    T[1] += (dz * r0.x - dx * r0.z) - r1.y;
                    T[2] += (dx * r0.y - dy * r0.x) - r1.z;
                } else {
                    F[0] += r0.x; F[1] += r0.y; F[2] += r0.z;
                    T[0] += r1.x; T[1] += r1.y; T[2] += r1.z;
                }
                U += real(0.5) * r0.w;
                // W^{ab} = r_ij^a F_ij^b with r_ij = -d: the same tensor seen from either side; half to each (R12)
                const real hx = real(-0.5) * dx, hy = real(-0.5) * dy, hz = real(-0.5) * dz;
                W[0] += hx * r0.x; W[1] += hx * r0.y; W[2] += hx * r0.z;
                W[3] += hy * r0.y; W[4] += hy * r0.z;
                W[5] += hz * r0.z;
            }
        }
    }
    for (int o = 1; o < lpp; o <<= 1) {  // combine the lanes of a particle (lpp divides 32: no particle straddles a warp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            F[a] += __shfl_xor_sync(0xffffffffu, F[a], o);
            T[a] += __shfl_xor_sync(0xffffffffu, T[a], o);
        }
        U += __shfl_xor_sync(0xffffffffu, U, o);
        if (virial) {
#pragma unroll
            for (int a = 0; a < 6; ++a) W[a] += __shfl_xor_sync(0xffffffffu, W[a], o);
        }
    }
    if (!lead) return;
    if (MODE != 2) {
        real4 f, t;
        f.x = F[0]; f.y = F[1]; f.z = F[2]; f.w = U;
        t.x = T[0]; t.y = T[1]; t.z = T[2]; t.w = real(0);
        force[i] = f;
        torque[i] = t;
        if (virial) {
#pragma unroll
            for (int a = 0; a < 6; ++a) virial[(size_t)i * 6 + a] = W[a];
        }
    }
    if (MODE >= 1) {
        // the state was asked for at the top (L2 prefetch): loading it only now keeps it out of the walk's registers
        d4 v = fa.vel[i], L = fa.ang[i], x, q, xb;
        const int sh = sid[i];
        if (MODE == 2) {
            x = fa.pos[i];
            q = fa.quat[i];
            xb = fa.pos_build[i];
        }
        const double hm = 0.5 * fa.dt / fa.mt.mass[sh];
        double vs[3] = {v.x, v.y, v.z}, Ls[3] = {L.x, L.y, L.z};
        const double Fs[3] = {(double)F[0], (double)F[1], (double)F[2]}, Ts[3] = {(double)T[0], (double)T[1], (double)T[2]};
        // (loops unrolled with predicates: static indices keep the state in registers)
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (a < fa.dim) vs[a] += hm * Fs[a];                                    // second half kick: the step is done
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (fa.dim == 3 || a == 2) Ls[a] += 0.5 * fa.dt * Ts[a];
        if (MODE == 2) {  // first half of the next step (the same arithmetic as k_kick_drift)
            double xs[3] = {x.x, x.y, x.z};
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (a < fa.dim) {
                    vs[a] += hm * Fs[a];
                    xs[a] += fa.dt * vs[a];
                    xs[a] -= fa.box.L[a] * rint(xs[a] * fa.box.invL[a]);
                }
            x.x = xs[0]; x.y = xs[1]; x.z = xs[2];
            fa.pos[i] = x;
            double dx = xs[0] - xb.x, dy = xs[1] - xb.y, dz = fa.dim == 3 ? xs[2] - xb.z : 0.0;
            dx -= fa.box.L[0] * rint(dx * fa.box.invL[0]);
            dy -= fa.box.L[1] * rint(dy * fa.box.invL[1]);
            dz -= fa.box.L[2] * rint(dz * fa.box.invL[2]);
            if (dx * dx + dy * dy + dz * dz > fa.half_skin2) *fa.raise = 1;
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (fa.dim == 3 || a == 2) Ls[a] += 0.5 * fa.dt * Ts[a];
            double qs[4] = {q.x, q.y, q.z, q.w};
            free_rotate(fa.dim, fa.mt.inertia[sh], Ls, fa.dt, qs);
            q.x = qs[0]; q.y = qs[1]; q.z = qs[2]; q.w = qs[3];
            fa.quat[i] = q;
        }
        v.x = vs[0]; v.y = vs[1]; v.z = vs[2];
        L.x = Ls[0]; L.y = Ls[1]; L.z = Ls[2];
        fa.vel[i] = v;
        fa.ang[i] = L;
    }
}

}  // namespace dem
