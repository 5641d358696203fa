// dem_kernels.cuh -- the CUDA kernels of libdem_b200 (sm_100a).  Host orchestration is in dem_lib.cu.
//
//   a3-a7 pair-feature kernel           k_pair          (FP32-ALU bound; dem_math.cuh holds the arithmetic)
//   a8  per-particle reduction          k_reduce        (warp-shuffle over 4 lanes per particle, no atomics)
// The neighbour-list kernels (a2) are in dem_list.cuh, the integrator (a9) in dem_integrate.cuh, the packed FP32 search
// kernels in dem_fast.cuh.
#pragma once
#include <cuda_runtime.h>

#include "dem_math.cuh"

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
    if ((threadIdx.x & 31) == 0) {
        if (c_eval) atomicAdd(a.counters + 0, (unsigned long long)c_eval);
        if (c_act) atomicAdd(a.counters + 1, (unsigned long long)c_act);
        if (c_deg) atomicAdd(a.counters + 2, (unsigned long long)c_deg);
        if (c_par) atomicAdd(a.counters + 3, (unsigned long long)c_par);
    }
}

// ---- a8: per-particle reduction -------------------------------------------------------------------------------------
// a particle's total is the sum over its neighbours.  4 lanes per particle walk its neighbour row, each
// reads the result records of its pairs (which side of the pair it is comes from `slot`, the pair's class from the
// class-major pair index; pairs whose record flag is 0 contribute nothing and have no record), and the 4 partial sums
// are combined with warp shuffles.  The summation order is fixed, so
// results are bit-reproducible from run to run.  With KICK the lane that stores the result also applies the second
// half kick of velocity Verlet (v += dt/2 F/m, L += dt/2 tau), which saves a pass over the state.
// `flags` (dem_step only, else null): flags[0] = "some particle left its skin in this step's drift" (k_kick_drift),
// flags[1] = halt, flags[2] = steps completed.  dem_step queues many steps before the host looks at the flags: with
// flags[0] set the list is stale, so the kernel changes nothing and raises halt, which turns every later
// k_kick_drift of the chunk into a no-op; otherwise it counts the step as completed (see step_t).
template <typename real, bool KICK>
__global__ void k_reduce(int N, const int* __restrict__ counts, const int* __restrict__ slot, int stride,
                         const int* __restrict__ sid, ClassTable ct, int nclass,
                         const typename vec4<real>::type* __restrict__ rec, const unsigned char* __restrict__ rflag,
                         typename vec4<real>::type* __restrict__ force,
                         typename vec4<real>::type* __restrict__ torque, real* __restrict__ virial,
                         int* __restrict__ flags, KickArgs ka) {
    typedef typename vec4<real>::type real4;
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (flags) {
        if (flags[0]) {
            if (gid == 0) flags[1] = 1;
            return;
        }
        if (gid == 0) flags[2] += 1;  // nothing in this kernel reads flags[2]
    }
    const int i = gid >> 2, sub = gid & 3;
    real F[3] = {0, 0, 0}, T[3] = {0, 0, 0}, U = 0, W[6] = {0, 0, 0, 0, 0, 0};
    if (i < N) {
        const int n = min(counts[i], stride);
        for (int k = sub; k < n; k += 4) {
            const int sl = slot[(size_t)i * stride + k];
            const int p = sl >> 1, side = sl & 1;
            int c = 0;
            while (c + 1 < nclass && p >= ct.pair_base[c + 1]) ++c;
            const int S = ct.slices[c];
            DEM_ASSERT(sl >= 0 && p < ct.pair_base[nclass] && p >= ct.pair_base[c]);
            const size_t r0i = (size_t)ct.rec_base[c] + (size_t)(p - ct.pair_base[c]) * S;
            const real4* r = rec + DEM_REC * r0i;
            for (int s = 0; s < S; ++s, r += DEM_REC) {
                if (!rflag[r0i + s]) continue;  // this (pair, slice) contributes nothing: no record was written
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
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
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
    if (i < N && sub == 0) {
        real4 f, t;
        f.x = F[0]; f.y = F[1]; f.z = F[2]; f.w = U;
        t.x = T[0]; t.y = T[1]; t.z = T[2]; t.w = real(0);
        force[i] = f;
        torque[i] = t;
        if (virial) {
#pragma unroll
            for (int a = 0; a < 6; ++a) virial[(size_t)i * 6 + a] = W[a];
        }
        if (KICK) {
            const double hm = ka.half_dt * ka.inv_mass[sid[i]];
            d4 v = ka.vel[i], L = ka.ang[i];
            v.x += hm * (double)F[0];
            v.y += hm * (double)F[1];
            if (ka.dim == 3) {
                v.z += hm * (double)F[2];
                L.x += ka.half_dt * (double)T[0];
                L.y += ka.half_dt * (double)T[1];
            }
            L.z += ka.half_dt * (double)T[2];
            ka.vel[i] = v;
            ka.ang[i] = L;
        }
    }
}

}  // namespace dem
