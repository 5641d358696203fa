// dem_step2d.cuh -- k_particle2d: the whole 2D hot path of a DEM_F32 context in ONE kernel per evaluation / time step.
//
// Eq. 2 has so few terms per pair (2 V E: 50 for pentagons) that the machinery of the 3D path -- a
// unique-pair work list, pose records, 48-byte pair records, a slot gather in the reduction -- moves more bytes than the
// terms justify (config 3: k_pair 64 us + k_reduce 36 us + k_kick_drift 28 us per step against ~15 us of HBM time for
// the state itself).  In 2D the paper's own decomposition is the better one on this machine: every particle evaluates
// its interaction with every neighbour of its (full) neighbour list, i.e. each unordered pair is evaluated twice, once
// from either side, and nothing is written but the particle's own totals.
//
//   gather   a warp owns 32 consecutive particles (one per lane).  Each lane walks its neighbour row, applies the
//            exact reach test (R10) in double and notes the neighbours inside the reach in a bit mask.
//   compact  the (owner lane, neighbour) entries of the warp are laid out owner-major in shared memory (exclusive
//            prefix of the lanes' counts), so that no lane idles on a neighbour that is out of reach or on a short row.
//   evaluate 32 entries at a time, one per lane: relative pose in FP64 rounded once to float (as everywhere in the
//            library), then every Eq. 2 term of the directed pair with the packed FP32 search (two vertices per lane
//            in the halves of 64-bit registers, FFMA2); the rare terms inside the candidate cutoff go through the
//            exact scalar routines of dem_math.cuh (WCA, force, torque), exactly as in the other kernels.
//   reduce   each entry's (F, tau, U, virial) goes to shared memory; the owner adds its entries in list order (fixed
//            order, no atomics: bit-reproducible) -- PAPER.md:65 "summed in shared memory".
//   finish   the owner stores F / tau / U / virial or, inside dem_step, goes on with the integrator (FinArgs: second half
//            kick, then first half kick, drift, rotation and skin test of the next step).  Because other warps still
//            read the old positions and orientations, the drift writes them to a second buffer (ping-pong).
#pragma once
#include "dem_fast.cuh"

namespace dem {

#define DEM_P2D_THREADS 128
#define DEM_P2D_MAXNB 64  // neighbours per particle the bit mask holds (the host falls back to the pair kernels beyond)

struct Particle2DArgs {
    int N, stride;
    const int* counts;
    const int* list;      // [N][stride] neighbour rows
    const int* sid;
    const f4* table;      // device shape table
    ShapeDev shape[DEM_MAX_SHAPES_K];
    int nshape, table_len;          // total length of the table in float4 (all shapes are staged)
    double rounding[DEM_MAX_SHAPES_K], circum[DEM_MAX_SHAPES_K];
    float eps, eps_par;
    int cull;             // exact per-vertex culling (dem_set_culling): a vertex farther than R + rc_search from the other
                          // particle's centre cannot be within the cutoff of any of its edges: its sweep is skipped
    BoxDev box;
    const void* pos;      // positions and orientations the forces are evaluated at: float[N][4] or double[N][4]
    const void* quat;
    f4* force;            // outputs (modes 0 and 1), may be null in mode 2
    f4* torque;
    float* virial;        // may be null
    unsigned long long* counters;  // [0] pairs evaluated, [1] active, [2] degenerate (unordered pairs: i < j); may be null
    unsigned long long* swept;     // [4] += vertex-edge terms swept (flop count of bench.py); may be null
    FinArgs fin;          // fin.pos / fin.quat: where the DRIFTED state is written (mode 2), never the buffers read above
};

template <typename PosT>
__global__ void __launch_bounds__(DEM_P2D_THREADS, 5) k_particle2d(const Particle2DArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // per warp: entries [32 * MAXNB] (owner << 8 | k, 16 bit), results [7][32] float, own poses [32] (x, y, cos, sin double)
    unsigned short* entries_all = reinterpret_cast<unsigned short*>(smem_raw);
    float* res_all = reinterpret_cast<float*>(entries_all + 4 * 32 * DEM_P2D_MAXNB);
    double* own_all = reinterpret_cast<double*>(res_all + 4 * 7 * 32);
    f4* sm = reinterpret_cast<f4*>(own_all + 4 * 32 * 4);
    for (int k = threadIdx.x; k < a.table_len; k += blockDim.x) sm[k] = a.table[k];
    __syncthreads();
    const FinArgs& fa = a.fin;
    if (fa.mode != 0 && fa.bail && *fa.bail) {  // the list went stale before this step (see FinArgs)
        if (blockIdx.x == 0 && threadIdx.x == 0 && fa.raise) *fa.raise = 1;
        return;
    }
    if (fa.mode != 0 && blockIdx.x == 0 && threadIdx.x == 0 && fa.done) *fa.done += 1;

    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned short* entries = entries_all + warp * 32 * DEM_P2D_MAXNB;
    float* res = res_all + warp * 7 * 32;
    double* own = own_all + warp * 32 * 4;
    const int i = (blockIdx.x * (DEM_P2D_THREADS / 32) + warp) * 32 + lane;
    const bool live = i < a.N;
    const PosT* pos = static_cast<const PosT*>(a.pos);
    const PosT* quat = static_cast<const PosT*>(a.quat);

    // ---- gather: own pose, reach test over the neighbour row -----------------------------------------------------------
    d4 xi, qi;
    xi.x = xi.y = xi.z = xi.w = 0.0;
    qi.x = 1.0; qi.y = qi.z = qi.w = 0.0;
    int si = 0, n = 0;
    if (live) {
        xi = load4d(pos, i);
        qi = load4d(quat, i);
        si = a.sid[i];
        n = a.counts[i];
        DEM_ASSERT(n <= DEM_P2D_MAXNB && n <= a.stride);
    }
    own[lane * 4 + 0] = xi.x; own[lane * 4 + 1] = xi.y; own[lane * 4 + 2] = qi.x; own[lane * 4 + 3] = qi.w;
    if (live && fa.mode >= 1) {  // the integrator's state is needed last: ask for it now
        asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.vel + i));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.ang + i));
        if (fa.mode == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(fa.pos_build + i));
    }
    const double rcw = 1.122462048309373;  // 2^(1/6)
    unsigned long long inreach = 0ull;
    const int* row = a.list + (size_t)i * a.stride;
    for (int k0 = 0; k0 < n; k0 += 4) {  // four neighbours at a time: their loads are in flight together
        int j[4];
        d4 xj[4];
        int sj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) j[u] = k0 + u < n ? row[k0 + u] : i;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            xj[u] = load4d(pos, j[u]);
            sj[u] = a.sid[j[u]];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            double dx = xj[u].x - xi.x, dy = xj[u].y - xi.y;
            dx -= a.box.L[0] * rint(dx * a.box.invL[0]);
            dy -= a.box.L[1] * rint(dy * a.box.invL[1]);
            const double reach = a.circum[si] + a.circum[sj[u]] + rcw * (a.rounding[si] + a.rounding[sj[u]]);
            if (k0 + u < n && dx * dx + dy * dy < reach * reach) inreach |= 1ull << (k0 + u);
        }
    }
    // ---- compact: owner-major entry list of the warp --------------------------------------------------------------------
    const int cnt = __popcll(inreach);
    int incl = cnt;
#pragma unroll
    for (int dlt = 1; dlt < 32; dlt <<= 1) {
        const int y = __shfl_up_sync(full, incl, dlt);
        if (lane >= dlt) incl += y;
    }
    const int off = incl - cnt, total = __shfl_sync(full, incl, 31);
    {
        int e = off;
        unsigned long long m = inreach;
        while (m) {
            const int k = __ffsll((long long)m) - 1;
            m &= m - 1ull;
            entries[e++] = (unsigned short)((lane << 8) | k);
        }
    }
    __syncwarp();

    // ---- evaluate + reduce: 32 entries per round, one per lane ---------------------------------------------------------
    float F[2] = {0.f, 0.f}, Tz = 0.f, U = 0.f, W[3] = {0.f, 0.f, 0.f};
    unsigned c_pairs = 0u, c_act = 0u, c_deg = 0u, c_swept = 0u;
    for (int base = 0; base < total; base += 32) {
        const int e = base + lane;
        float out[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (e < total) {
            const int ow = entries[e] >> 8, k = entries[e] & 0xff;
            const int io = i - lane + ow;
            const int j = a.list[(size_t)io * a.stride + k];
            const int so = a.sid[io], sj = a.sid[j];
            const d4 xj = load4d(pos, j), qj = load4d(quat, j);
            double d[3] = {xj.x - own[ow * 4 + 0], xj.y - own[ow * 4 + 1], 0.0};
            d[0] -= a.box.L[0] * rint(d[0] * a.box.invL[0]);
            d[1] -= a.box.L[1] * rint(d[1] * a.box.invL[1]);
            // relative pose in FP64, rounded once: rotation matrices of (w, 0, 0, z) are [[c, -s], [s, c]], c = 1 - 2 z^2,
            // s = 2 w z; R = R_i^T R_j, t = R_i^T d (the 2D case of pair_pose)
            float Mi[9], R[9], t[3];
            {
                const double wi = own[ow * 4 + 2], zi = own[ow * 4 + 3];
                const double ci = 1.0 - 2.0 * zi * zi, sni = 2.0 * wi * zi;
                const double cj = 1.0 - 2.0 * qj.w * qj.w, snj = 2.0 * qj.x * qj.w;
                const double cr = ci * cj + sni * snj, sr = ci * snj - sni * cj;
                R[0] = (float)cr; R[1] = (float)-sr; R[2] = 0.f; R[3] = (float)sr; R[4] = (float)cr; R[5] = 0.f;
                R[6] = R[7] = 0.f; R[8] = 1.f;
                t[0] = (float)(ci * d[0] + sni * d[1]); t[1] = (float)(ci * d[1] - sni * d[0]); t[2] = 0.f;
                Mi[0] = (float)ci; Mi[1] = (float)-sni; Mi[2] = 0.f; Mi[3] = (float)sni; Mi[4] = (float)ci; Mi[5] = 0.f;
                Mi[6] = Mi[7] = 0.f; Mi[8] = 1.f;
            }
            // shapes of the directed pair: A = the owner's (working frame), B = the neighbour's
            ShapeView<float> A, B;
            const ShapeDev &sa = a.shape[so], &sb = a.shape[sj];
            A.nv = sa.nv; A.ne = sa.ne; A.nf = 0; A.V = sm + sa.off; A.E = A.V + A.nv; A.F = A.FE = A.OE = nullptr;
            B.nv = sb.nv; B.ne = sb.ne; B.nf = 0; B.V = sm + sb.off; B.E = B.V + B.nv; B.F = B.FE = B.OE = nullptr;
            const double sigma = a.rounding[so] + a.rounding[sj];
            PairConst<float> pc;
            pc.rc2 = (float)(1.2599210498948732 * sigma * sigma);  // 2^(1/3) sigma^2
            pc.sig2 = (float)(sigma * sigma);
            pc.eps = a.eps;
            pc.eps_par = a.eps_par;
            pc.degen2 = (float)((1e-6 * sigma) * (1e-6 * sigma));
            const double rcs = rcw * sigma * (1.0 + 1e-3);  // candidate cutoff of the packed search
            const float nrc2 = -(float)(rcs * rcs);
            // culling radii: a vertex of j can only reach an edge of the owner from within R_owner + rc_search of the
            // owner's centre (|p| in the owner's frame), and the other way round (|v - t| = the vertex seen from j's centre)
            const float big = 3.0e38f;
            const float cull_a2 = a.cull ? (float)((a.circum[so] + rcs) * (a.circum[so] + rcs)) : big;
            const float cull_b2 = a.cull ? (float)((a.circum[sj] + rcs) * (a.circum[sj] + rcs)) : big;
            PairAcc<float> acc;
            acc.F[0] = acc.F[1] = acc.F[2] = acc.T[0] = acc.T[1] = acc.T[2] = acc.u = 0.f;
            acc.nactive = acc.ndegen = acc.npar = 0u;
            // The sweeps only note candidates (side, vertex, edge: one per term inside the candidate cutoff) in a small
            // per-lane list; the exact scalar routines run on them afterwards, in one place.
            // (four named registers, filled and emptied with static moves: an indexed array would live in local memory)
            unsigned cand0 = 0u, cand1 = 0u, cand2 = 0u, cand3 = 0u;
            int ncand = 0;
            auto eval_cand = [&](unsigned c0) {
                const int sd_ = (int)(c0 >> 31), o_ = (int)((c0 >> 12) & 0x7ffffu), k_ = (int)(c0 & 0xfffu);
                if (sd_ == 0) {
                    const f4 v = B.V[o_];
                    float p[3];
                    vertex_to_i<float>(v.x, v.y, 0.f, R, t, p);
                    term_ve_own<float>(A, k_, p[0], p[1], pc, acc);
                } else {
                    const f4 v = A.V[o_];
                    float p[3];
                    vertex_to_j<float>(v.x, v.y, 0.f, R, t, p);
                    term_ve_other<float>(B, k_, v.x, v.y, p[0], p[1], R, pc, acc);
                }
            };
            auto note = [&](int side, int o, int kk) {
                if (ncand == 4) {  // list full (rare): evaluate the oldest entry now
                    const unsigned c0 = cand0;
                    cand0 = cand1; cand1 = cand2; cand2 = cand3;
                    ncand = 3;
                    eval_cand(c0);
                }
                const unsigned v = ((unsigned)side << 31) | ((unsigned)o << 12) | (unsigned)kk;
                if (ncand == 0) cand0 = v;
                else if (ncand == 1) cand1 = v;
                else if (ncand == 2) cand2 = v;
                else cand3 = v;
                ++ncand;
            };
#pragma unroll 1
            for (int side = 0; side < 2; ++side) {
                // side 0, first sum of Eq. 2: vertices of j (in the owner's frame) against the owner's edges;
                // side 1, second sum: the owner's vertices (in j's frame) against the edges of j
                const ShapeView<float>& Out = side == 0 ? B : A;
                const ShapeView<float>& In = side == 0 ? A : B;
                const float c2 = side == 0 ? cull_a2 : cull_b2;
                unsigned long long surv = 0ull;  // vertices that survive the cull (all of them without culling)
                for (int o = 0; o < Out.nv; ++o) {
                    const f4 v = Out.V[o];
                    float x, y;
                    if (side == 0) { x = R[0] * v.x + R[1] * v.y + t[0]; y = R[3] * v.x + R[4] * v.y + t[1]; }
                    else { x = v.x - t[0]; y = v.y - t[1]; }
                    surv |= (unsigned long long)(x * x + y * y < c2) << o;
                }
                c_swept += (unsigned)(__popcll(surv) * In.ne);
                // With culling one or two vertices survive per side: a packed pair of them would mostly carry a
                // duplicate, so the survivors are swept one at a time with scalar arithmetic (without culling the packed
                // sweep below takes them two at a time)
                if (a.cull) {
                    while (surv) {
                        const int o0 = __ffsll((long long)surv) - 1;
                        surv &= surv - 1ull;
                        const f4 va = Out.V[o0];
                        float pa[3];
                        if (side == 0) vertex_to_i<float>(va.x, va.y, 0.f, R, t, pa);
                        else vertex_to_j<float>(va.x, va.y, 0.f, R, t, pa);
                        for (int kk = 0; kk < In.ne; ++kk) {
                            const f4 e0 = In.E[2 * kk], e1 = In.E[2 * kk + 1];
                            const float sd = e0.z * pa[1] - e0.w * pa[0] + e1.y, am = e0.z * pa[0] + e0.w * pa[1] + e1.z;
                            const float ex = fmaxf(fabsf(am) - e1.w, 0.f);
                            if (sd * sd + ex * ex + nrc2 < 0.f) note(side, o0, kk);
                        }
                    }
                }
                while (surv) {  // two surviving vertices per packed sweep
                    const int o0 = __ffsll((long long)surv) - 1;
                    surv &= surv - 1ull;
                    const int o1 = surv ? __ffsll((long long)surv) - 1 : o0;
                    surv &= surv - 1ull;
                    const f4 va = Out.V[o0], vb = Out.V[o1];
                    float pa[3], pb[3];
                    if (side == 0) {
                        vertex_to_i<float>(va.x, va.y, 0.f, R, t, pa);
                        vertex_to_i<float>(vb.x, vb.y, 0.f, R, t, pb);
                    } else {
                        vertex_to_j<float>(va.x, va.y, 0.f, R, t, pa);
                        vertex_to_j<float>(vb.x, vb.y, 0.f, R, t, pb);
                    }
                    const u64 px = pk(pa[0], pb[0]), py = pk(pa[1], pb[1]);
                    for (int kk = 0; kk < In.ne; ++kk) {
                        u64 sd, exc;
                        edge2_eval(In.E[2 * kk], In.E[2 * kk + 1], px, py, sd, exc);
                        float lo, hi;
                        upk(fma2(exc, exc, fma2(sd, sd, bc(nrc2))), lo, hi);
                        if (fminf(lo, hi) < 0.f) {
                            if (lo < 0.f) note(side, o0, kk);
                            if (hi < 0.f && o1 != o0) note(side, o1, kk);
                        }
                    }
                }
            }
#pragma unroll 1
            for (int c = 0; c < ncand; ++c) {  // oldest first
                const unsigned c0 = cand0;
                cand0 = cand1; cand1 = cand2; cand2 = cand3;
                eval_cand(c0);
            }
            if (acc.nactive) {
                float o10[10];
                pair_finish<float>(Mi, t, acc.F, acc.T, acc.u, o10);
                out[0] = o10[0]; out[1] = o10[1]; out[2] = o10[5]; out[3] = 0.5f * o10[9];
                // W^{ab} = r_ij^a F_ij^b with r_ij = -d, half to each particle (R12)
                const float hx = -0.5f * (float)d[0], hy = -0.5f * (float)d[1];
                out[4] = hx * o10[0]; out[5] = hx * o10[1]; out[6] = hy * o10[1];
            }
            if (io < j) {  // counters are per unordered pair
                c_pairs += 1u;
                c_act += acc.nactive;
                c_deg += acc.ndegen;
            }
        }
#pragma unroll
        for (int c = 0; c < 7; ++c) res[c * 32 + lane] = out[c];
        __syncwarp();
        // the owner adds its entries of this round, in list order
        const int b = max(off, base), en = min(off + cnt, base + 32);
        for (int x = b; x < en; ++x) {
            const int r = x - base;
            F[0] += res[0 * 32 + r]; F[1] += res[1 * 32 + r]; Tz += res[2 * 32 + r]; U += res[3 * 32 + r];
            W[0] += res[4 * 32 + r]; W[1] += res[5 * 32 + r]; W[2] += res[6 * 32 + r];
        }
        __syncwarp();
    }
    if (a.counters || a.swept) {
        const unsigned s0 = __reduce_add_sync(full, c_pairs), s1 = __reduce_add_sync(full, c_act),
                       s2 = __reduce_add_sync(full, c_deg), s3 = __reduce_add_sync(full, c_swept);
        if (lane == 0) {
            if (a.counters) {
                if (s0) atomicAdd(a.counters + 0, (unsigned long long)s0);
                if (s1) atomicAdd(a.counters + 1, (unsigned long long)s1);
                if (s2) atomicAdd(a.counters + 2, (unsigned long long)s2);
                if (s3) atomicAdd(a.counters + 4, (unsigned long long)(s3 >> 1));  // each pair's terms are swept twice
            }
            if (a.swept && s3) atomicAdd(a.swept, (unsigned long long)(s3 >> 1));
        }
    }
    if (!live) return;

    // ---- finish --------------------------------------------------------------------------------------------------------
    if (fa.mode != 2) {
        f4 f, tq;
        f.x = F[0]; f.y = F[1]; f.z = 0.f; f.w = U;
        tq.x = tq.y = 0.f; tq.z = Tz; tq.w = 0.f;
        a.force[i] = f;
        a.torque[i] = tq;
        if (a.virial) {
            float* w = a.virial + (size_t)i * 6;
            w[0] = W[0]; w[1] = W[1]; w[2] = 0.f; w[3] = W[2]; w[4] = 0.f; w[5] = 0.f;
        }
    }
    if (fa.mode >= 1) {
        d4 v = fa.vel[i], L = fa.ang[i];
        const double hm = 0.5 * fa.dt / fa.mt.mass[si];
        v.x += hm * (double)F[0];  // second half kick: the step is done
        v.y += hm * (double)F[1];
        L.z += 0.5 * fa.dt * (double)Tz;
        if (fa.mode == 2) {  // first half of the next step (the arithmetic of k_kick_drift); state goes to the other buffer
            const d4 xb = fa.pos_build[i];
            v.x += hm * (double)F[0];
            v.y += hm * (double)F[1];
            d4 x = xi;
            x.x += fa.dt * v.x;
            x.y += fa.dt * v.y;
            x.x -= fa.box.L[0] * rint(x.x * fa.box.invL[0]);
            x.y -= fa.box.L[1] * rint(x.y * fa.box.invL[1]);
            fa.pos[i] = x;
            double dx = x.x - xb.x, dy = x.y - xb.y;
            dx -= fa.box.L[0] * rint(dx * fa.box.invL[0]);
            dy -= fa.box.L[1] * rint(dy * fa.box.invL[1]);
            if (dx * dx + dy * dy > fa.half_skin2) *fa.raise = 1;
            L.z += 0.5 * fa.dt * (double)Tz;
            double Ls[3] = {L.x, L.y, L.z}, qs[4] = {qi.x, qi.y, qi.z, qi.w};
            free_rotate(2, fa.mt.inertia[si], Ls, fa.dt, qs);
            d4 q;
            q.x = qs[0]; q.y = qs[1]; q.z = qs[2]; q.w = qs[3];
            fa.quat[i] = q;
        }
        fa.vel[i] = v;
        fa.ang[i] = L;
    }
}

static inline size_t particle2d_smem(int table_len) {
    return sizeof(unsigned short) * 4 * 32 * DEM_P2D_MAXNB + sizeof(float) * 4 * 7 * 32 + sizeof(double) * 4 * 32 * 4 +
           sizeof(f4) * (size_t)table_len;
}

}  // namespace dem
