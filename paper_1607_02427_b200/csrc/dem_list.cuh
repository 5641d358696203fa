// dem_list.cuh -- a2: cell list, full neighbour list and the unique-pair work list (HBM / latency bound).
//   k_bin, k_scan_block, k_scan_add, k_place, k_sort_cells, k_gather_sorted, k_neigh, k_copy_rows,
//   k_pair_count, k_pair_fill, k_slot_back.   Included by dem_lib.cu only (the kernels are not templates).
#pragma once
#include "dem_kernels.cuh"

namespace dem {

// ---- a2: cell list --------------------------------------------------------------------------------------------------
template <typename PosT>
__global__ void k_bin(const PosT* __restrict__ pos, int N, BoxDev box, GridDev g, int* __restrict__ cell_of,
                      int* __restrict__ cell_cnt, int* __restrict__ rank) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const d4 x = load4d(pos, i);
    const double xs[3] = {x.x, x.y, x.z};
    int c[3] = {0, 0, 0};
    for (int a = 0; a < box.dim; ++a) {
        double f = xs[a] / box.L[a] + 0.5;
        f -= floor(f);
        int ca = (int)(f * g.nc[a]);
        c[a] = min(max(ca, 0), g.nc[a] - 1);
    }
    const int cell = (c[2] * g.nc[1] + c[1]) * g.nc[0] + c[0];
    cell_of[i] = cell;
    rank[i] = atomicAdd(&cell_cnt[cell], 1);
}

// exclusive scan of int data[n] in place, blocks of 1024; block totals to sums[blockIdx]
__global__ void k_scan_block(int* __restrict__ data, int n, int* __restrict__ sums) {
    __shared__ int warp_tot[32];
    const int i = blockIdx.x * 1024 + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int v = i < n ? data[i] : 0;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_tot[w] = x;
    __syncthreads();
    if (w == 0) {
        int t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += y;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    const int base = w ? warp_tot[w - 1] : 0;
    if (i < n) data[i] = base + x - v;
    if (threadIdx.x == 1023 && sums) sums[blockIdx.x] = base + x;
}
__global__ void k_scan_add(int* __restrict__ data, int n, const int* __restrict__ sums) {
    const int i = blockIdx.x * 1024 + threadIdx.x;
    if (i < n) data[i] += sums[blockIdx.x];
}

__global__ void k_place(int N, const int* __restrict__ cell_of, const int* __restrict__ rank,
                        const int* __restrict__ cell_start, int* __restrict__ order) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) order[cell_start[cell_of[i]] + rank[i]] = i;
}

// The atomic ranks above depend on scheduling; sorting each cell's few members by particle index makes the cell
// list, hence the neighbour rows, the pair list and every summation order, identical from run to run.
__global__ void k_sort_cells(int ncell, const int* __restrict__ cell_start, int* __restrict__ order) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int b = cell_start[c], e = cell_start[c + 1];
    for (int m = b + 1; m < e; ++m) {
        const int v = order[m];
        int k = m - 1;
        while (k >= b && order[k] > v) {
            order[k + 1] = order[k];
            --k;
        }
        order[k + 1] = v;
    }
}

template <typename PosT>
__global__ void k_gather_sorted(const PosT* __restrict__ pos, int N, const int* __restrict__ order, d4* __restrict__ xs) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < N) xs[s] = load4d(pos, order[s]);
}

// One thread per particle (in cell order, so a warp's candidate cells overlap in L1/L2).  Candidates from the
// 3^dim adjacent cells; the predicate is the definition (R13) in double.  Rows are written for the ORIGINAL index.
__global__ void k_neigh(int N, BoxDev box, GridDev g, double rc2, const int* __restrict__ order,
                        const int* __restrict__ cell_of, const int* __restrict__ cell_start, const d4* __restrict__ xs,
                        int stride, int* __restrict__ counts, int* __restrict__ list, int* __restrict__ max_count) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int i = order[s];
    const d4 xi = xs[s];
    int cell = cell_of[i];
    const int cx = cell % g.nc[0];
    cell /= g.nc[0];
    const int cy = cell % g.nc[1], cz = cell / g.nc[1];
    // per axis: all cells if there are fewer than 3, else the three adjacent ones (wrapped)
    const int nx = g.nc[0] < 3 ? g.nc[0] : 3, ny = g.nc[1] < 3 ? g.nc[1] : 3, nz = g.nc[2] < 3 ? g.nc[2] : 3;
    int cnt = 0;
    int* row = list + (size_t)i * stride;
    for (int iz = 0; iz < nz; ++iz) {
        const int z = g.nc[2] < 3 ? iz : (cz + iz - 1 + g.nc[2]) % g.nc[2];
        for (int iy = 0; iy < ny; ++iy) {
            const int y = g.nc[1] < 3 ? iy : (cy + iy - 1 + g.nc[1]) % g.nc[1];
            for (int ix = 0; ix < nx; ++ix) {
                const int x = g.nc[0] < 3 ? ix : (cx + ix - 1 + g.nc[0]) % g.nc[0];
                const int c2 = (z * g.nc[1] + y) * g.nc[0] + x;
                const int b = cell_start[c2], e = cell_start[c2 + 1];
                for (int m = b; m < e; ++m) {
                    if (m == s) continue;
                    const d4 xj = xs[m];
                    const double dx = min_image_1(xi.x, xj.x, box.L[0], box.invL[0]);
                    const double dy = min_image_1(xi.y, xj.y, box.L[1], box.invL[1]);
                    const double dz = box.dim == 3 ? min_image_1(xi.z, xj.z, box.L[2], box.invL[2]) : 0.0;
                    if (norm2_fma(dx, dy, dz) < rc2) {
                        if (cnt < stride) row[cnt] = order[m];
                        ++cnt;
                    }
                }
            }
        }
    }
    counts[i] = cnt;
    if (cnt > 0) atomicMax(max_count, cnt);
}

__global__ void k_copy_rows(int N, const int* __restrict__ counts, const int* __restrict__ list, int stride,
                            int* __restrict__ out, int out_stride) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * out_stride) return;
    const int i = (int)(t / out_stride), k = (int)(t % out_stride);
    out[t] = k < counts[i] ? list[(size_t)i * stride + k] : -1;
}

// ---- unique-pair work list ------------------------------------------------------------------------------------------
// Each unordered neighbour pair {i, j} is evaluated ONCE (the method's own cost: Eq. 1/2 per pair).  The pair list is
// class-major (class = unordered pair of shape ids) so that a warp of the pair kernel runs 32 pairs with identical
// loop bounds and identical (warp-uniform) shape-table addresses.  `slot` tells each side where its pair's result
// records live, so that the reduction needs no atomics.
__global__ void k_pair_count(int N, const int* __restrict__ counts, const int* __restrict__ list, int stride,
                             const int* __restrict__ sid, ClassTable ct, int nclass, int nshape, int* __restrict__ pcnt,
                             int* __restrict__ bad_shape) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int loc[DEM_MAX_CLASSES];
    for (int c = 0; c < nclass; ++c) loc[c] = 0;
    const int si = sid[i];
    // a shape id outside the registered shapes would index the class table out of bounds here and in every kernel that
    // follows: flag it (dem_build_neighbors returns DEM_EINVAL) and list no pair for it
    const bool ok = si >= 0 && si < nshape;
    if (!ok) *bad_shape = 1;
    const int n = ok ? min(counts[i], stride) : 0;
    for (int k = 0; k < n; ++k) {
        const int j = list[(size_t)i * stride + k];
        if (j > i) {
            const int sj = sid[j];
            if (sj >= 0 && sj < nshape) loc[ct.lut[si][sj]]++;
        }
    }
    for (int c = 0; c < nclass; ++c) pcnt[(size_t)c * N + i] = loc[c];
}

__global__ void k_pair_fill(int N, const int* __restrict__ counts, const int* __restrict__ list, int stride,
                            const int* __restrict__ sid, ClassTable ct, int nclass, const int* __restrict__ poff,
                            int2* __restrict__ pairs, int* __restrict__ slot) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int loc[DEM_MAX_CLASSES];
    for (int c = 0; c < nclass; ++c) loc[c] = poff[(size_t)c * N + i];
    const int si = sid[i];
    const int n = min(counts[i], stride);
    for (int k = 0; k < n; ++k) {
        const int j = list[(size_t)i * stride + k];
        if (j > i) {
            const int sj = sid[j];
            const int p = loc[ct.lut[si][sj]]++;
            DEM_ASSERT(p >= 0 && p < ct.pair_base[nclass]);
            const bool i_first = si <= sj;  // the pair's first particle is the one with the smaller shape id
            pairs[p] = i_first ? make_int2(i, j) : make_int2(j, i);
            slot[(size_t)k * N + i] = 2 * p + (i_first ? 0 : 1);  // neighbour-major: [stride][N]
        }
    }
}

__global__ void k_slot_back(int N, const int* __restrict__ counts, const int* __restrict__ list, int stride,
                            const int* __restrict__ sid, ClassTable ct, const int* __restrict__ poff,
                            int* __restrict__ slot) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int si = sid[i];
    const int n = min(counts[i], stride);
    for (int k = 0; k < n; ++k) {
        const int j = list[(size_t)i * stride + k];
        if (j < i) {  // the pair is owned by j: find its position among j's owned pairs of the same class
            const int sj = sid[j];
            const int c = ct.lut[sj][si];
            const int nj = min(counts[j], stride);
            int r = 0;
            for (int m = 0; m < nj; ++m) {
                const int q = list[(size_t)j * stride + m];
                if (q == i) break;
                if (q > j && ct.lut[sj][sid[q]] == c) ++r;
            }
            const int p = poff[(size_t)c * N + j] + r;
            DEM_ASSERT(r < nj && p >= ct.pair_base[c] && p < ct.pair_base[c + 1]);
            const bool j_first = sj <= si;
            slot[(size_t)k * N + i] = 2 * p + (j_first ? 1 : 0);
        }
    }
    for (int k = n; k < stride; ++k) slot[(size_t)k * N + i] = -1;  // end of the row (k_finish stops there)
}

}  // namespace dem
