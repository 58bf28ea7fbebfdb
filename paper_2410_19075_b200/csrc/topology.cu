// Topology builder: emits lattice offset tables, validated CSR or the seeded random
// fixed-in-degree graph on the device, and expands any topology to canonical CSR rows
// (parity hook).  Integer-only; results are bit-exact by construction.
// Rules: PAPER.md:299-301 (ring), :309-313 (disc / ball, index map), :147 (orientation);
// random graph: DESIGN.md reading R8.
#include <stdlib.h>

#include "oscnet_internal.cuh"

namespace oscnet {

int32_t topo_lattice_noff(int ndim, int P, int include_self) {
    int Pz = ndim >= 3 ? P : 0, Py = ndim >= 2 ? P : 0, c = 0;
    for (int dz = -Pz; dz <= Pz; ++dz)
        for (int dy = -Py; dy <= Py; ++dy)
            for (int dx = -P; dx <= P; ++dx)
                if (dx * dx + dy * dy + dz * dz <= P * P) ++c;
    return include_self ? c : c - 1;
}

// One block enumerates the (2P+1)^ndim cube in (dz,dy,dx) order; every thread tests a strip of
// candidates, an exclusive scan over the per-thread counts gives the output slots.
__global__ void lattice_offsets_kernel(int ndim, int P, int include_self, int32_t* off, int32_t* count) {
    __shared__ int cnt[256];
    __shared__ int base[257];
    const int w = 2 * P + 1;
    const int Wy = ndim >= 2 ? w : 1, Wz = ndim >= 3 ? w : 1;
    const int total = w * Wy * Wz;
    const int per = (total + blockDim.x - 1) / blockDim.x;
    const int b = threadIdx.x * per, e = min(total, b + per);
    auto inside = [&](int c, int* dx, int* dy, int* dz) {
        *dx = c % w - P;
        *dy = ndim >= 2 ? (c / w) % w - P : 0;
        *dz = ndim >= 3 ? c / (w * w) - P : 0;
        if (*dx * *dx + *dy * *dy + *dz * *dz > P * P) return false;
        if (*dx == 0 && *dy == 0 && *dz == 0 && !include_self) return false;
        return true;
    };
    int c0 = 0, dx, dy, dz;
    for (int c = b; c < e; ++c) c0 += inside(c, &dx, &dy, &dz) ? 1 : 0;
    cnt[threadIdx.x] = c0;
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0;
        for (int t = 0; t < (int)blockDim.x; ++t) { base[t] = s; s += cnt[t]; }
        base[blockDim.x] = s;
        *count = s;
    }
    __syncthreads();
    int pos = base[threadIdx.x];
    for (int c = b; c < e; ++c)
        if (inside(c, &dx, &dy, &dz)) {
            off[3 * pos] = dx; off[3 * pos + 1] = dy; off[3 * pos + 2] = dz;
            ++pos;
        }
}

// CSR validation: row_ptr[0]==0, monotone, row_ptr[n]==nnz, 0 <= col < n.
__global__ void csr_validate_kernel(const int64_t* row_ptr, const int32_t* col_idx, int64_t n,
                                    int64_t nnz, int32_t* flag) {
    int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    if (tid == 0 && (row_ptr[0] != 0 || row_ptr[n] != nnz)) atomicOr(flag, 1);
    for (int64_t i = tid; i < n; i += stride)
        if (row_ptr[i + 1] < row_ptr[i]) atomicOr(flag, 1);
    for (int64_t e = tid; e < nnz; e += stride) {
        int32_t j = col_idx[e];
        if (j < 0 || (int64_t)j >= n) atomicOr(flag, 2);
    }
}

__global__ void csr_degree_kernel(const int64_t* row_ptr, int64_t n, int32_t* flag) {
    // flag[1] = degree of row 0; flag[2] |= 1 if any row differs
    int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int64_t d0 = row_ptr[1] - row_ptr[0];
    if (tid == 0) flag[1] = (int32_t)d0;
    for (int64_t i = tid; i < n; i += (int64_t)gridDim.x * blockDim.x)
        if (row_ptr[i + 1] - row_ptr[i] != d0) atomicOr(flag + 2, 1);
}

// splitmix64 finaliser (public-domain algorithm, restated; reading R8)
__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

// One thread per row.  The row is kept sorted while it is filled (binary search for the
// duplicate test, shift-insert), so it ends sorted ascending with k distinct sources != i.
__global__ void random_indegree_kernel(int64_t n, int32_t k, uint64_t seed, int32_t* col_idx) {
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        int32_t* row = col_idx + i * (int64_t)k;
        const uint64_t hi = mix64(seed + G * (uint64_t)(i + 1));
        int have = 0;
        for (uint64_t t = 0; have < k; ++t) {
            uint64_t hsh = mix64(hi + G * (t + 1));
            uint64_t j = __umul64hi(hsh, (uint64_t)(n - 1));
            if (j >= (uint64_t)i) j += 1;
            int32_t jj = (int32_t)j;
            int lo = 0, hi_ = have;  // first position with row[pos] >= jj
            while (lo < hi_) {
                int mid = (lo + hi_) >> 1;
                if (row[mid] < jj) lo = mid + 1; else hi_ = mid;
            }
            if (lo < have && row[lo] == jj) continue;
            for (int q = have; q > lo; --q) row[q] = row[q - 1];
            row[lo] = jj;
            ++have;
        }
    }
}

__global__ void uniform_row_ptr_kernel(int64_t* row_ptr, int64_t rows, int64_t k) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i <= rows;
         i += (int64_t)gridDim.x * blockDim.x)
        row_ptr[i] = i * k;
}

// Expansion of ring / lattice rows to canonical CSR: one thread per row writes its
// neighbours and insertion-sorts them in place.
__global__ void expand_rows_kernel(TopoView tv, int64_t n, int64_t row_begin, int64_t row_count,
                                   int32_t deg, int32_t* col_idx) {
    for (int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; r < row_count;
         r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = row_begin + r;
        int32_t* row = col_idx + r * (int64_t)deg;
        int have = 0;
        auto put = [&](int64_t j) {
            int32_t jj = (int32_t)j;
            int q = have;
            while (q > 0 && row[q - 1] > jj) { row[q] = row[q - 1]; --q; }
            row[q] = jj;
            ++have;
        };
        if (tv.kind == NET_TOPO_RING) {
            const int64_t rn = tv.ring_n, base = i / rn * rn;
            for (int d = -tv.P; d <= tv.P; ++d) {
                if (d == 0 && !tv.include_self) continue;
                int64_t j = i - base + d;
                if (j < 0) j += rn;
                if (j >= rn) j -= rn;
                put(base + j);
            }
        } else {
            const int64_t rbase = i / tv.ring_n * tv.ring_n, il = i - rbase;      // replica of a batch
            int x = (int)(il % tv.nx);
            int64_t q = il / tv.nx;
            int y = (int)(q % tv.ny), z = (int)(q / tv.ny);
            for (int o = 0; o < tv.noff; ++o) {
                int xx = x + tv.off[3 * o], yy = y + tv.off[3 * o + 1], zz = z + tv.off[3 * o + 2];
                xx += (xx < 0) ? tv.nx : 0; xx -= (xx >= tv.nx) ? tv.nx : 0;
                yy += (yy < 0) ? tv.ny : 0; yy -= (yy >= tv.ny) ? tv.ny : 0;
                zz += (zz < 0) ? tv.nz : 0; zz -= (zz >= tv.nz) ? tv.nz : 0;
                put(rbase + ((int64_t)zz * tv.ny + yy) * tv.nx + xx);
            }
        }
    }
}

// Ring rows in canonical order without sorting, one thread per (row, slot): the sequence
// j = i+d, d = -P..P, is ascending except at the single wrap point, so the sorted row is a
// rotation of it.  (Rows of config 2 have 45 874 entries: an in-thread sort is hopeless.)
__global__ void expand_ring_kernel(int64_t n, int32_t P, int32_t include_self, int64_t row_begin,
                                   int64_t row_count, int32_t deg, int32_t* col_idx) {
    const int64_t total = row_count * (int64_t)deg;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < total;
         e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = e / deg;
        const int32_t q = (int32_t)(e - r * deg);
        const int64_t gi = row_begin + r, base = gi / n * n, i = gi - base;   // n = ring period; i local to its ring
        int64_t d = (int64_t)q - P;
        if (!include_self && d >= 0) d += 1;
        int64_t j = i + d;
        int64_t pos;
        if (i - P < 0) {                      // the first c entries wrap to the top of the range
            const int64_t c = P - i;
            pos = q < c ? deg - c + q : q - c;
        } else if (i + P > n - 1) {           // the last c entries wrap to the bottom
            const int64_t c = i + P - (n - 1);
            pos = q >= deg - c ? q - (deg - c) : q + c;
        } else pos = q;
        if (j < 0) j += n;
        if (j >= n) j -= n;
        col_idx[r * (int64_t)deg + pos] = (int32_t)(base + j);
    }
}

// rn = rows of one replica (the arrays describe one replica; a batch repeats them block-diagonally)
__global__ void copy_rows_kernel(const int64_t* row_ptr, const int32_t* col_idx, int64_t row_begin,
                                 int64_t row_count, int64_t* out_ptr, int32_t* out_idx, int64_t rn) {
    const int64_t nnz1 = row_ptr[rn];
    auto gptr = [&](int64_t i) { return (i / rn) * nnz1 + row_ptr[i % rn]; };     // row_ptr of the whole batch
    const int64_t base = gptr(row_begin);
    int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t r = tid; r <= row_count; r += stride) out_ptr[r] = gptr(row_begin + r) - base;
    for (int64_t r = tid; r < row_count; r += stride) {
        const int64_t i = row_begin + r, rep = i / rn, il = i % rn;
        int32_t* dst = out_idx + (gptr(i) - base);
        for (int64_t e = row_ptr[il]; e < row_ptr[il + 1]; ++e) dst[e - row_ptr[il]] = (int32_t)(rep * rn + col_idx[e]);
    }
}

// NET_TOPO_COMPRESSED: degrees of a row range (EXTRACT counts), then the rows themselves, sorted
__global__ void compressed_degree_kernel(TopoView tv, int64_t row_begin, int64_t row_count, int64_t* out_ptr) {
    for (int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; r <= row_count; r += (int64_t)gridDim.x * blockDim.x)
        out_ptr[r] = r == 0 ? 0 : tv.cmp_deg[tv.cmp_c[row_begin + r - 1]];
}

// in-place inclusive scan of ptr[0..count] by one CTA (count + 1 values; ptr[0] = 0)
__global__ void __launch_bounds__(1024) scan_i64_kernel(int64_t* ptr, int64_t count) {
    __shared__ int64_t wsum[32];
    __shared__ int64_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int64_t base = 0; base <= count; base += 1024) {
        const int64_t s = base + threadIdx.x;
        int64_t v = s <= count ? ptr[s] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int64_t u = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += u;
        }
        if (lane == 31) wsum[warp] = v;
        __syncthreads();
        int64_t off = carry_s;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        v += off;
        if (s <= count) ptr[s] = v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = v;
        __syncthreads();
    }
}

__global__ void compressed_expand_kernel(TopoView tv, int64_t n, int64_t row_begin, int64_t row_count,
                                         const int64_t* out_ptr, int32_t* col_idx) {
    for (int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; r < row_count; r += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = row_begin + r;
        int32_t* row = col_idx + out_ptr[r];
        const int c = tv.cmp_c[i];
        int64_t b = tv.cmp_dptr[c];
        const int64_t be = tv.cmp_dptr[c + 1];
        int a = 0, have = 0;
        // positions p ascend; (p + i) mod n ascends too except at the single wrap: entries that wrap
        // (p + i >= n) are smaller than all that do not, so they are written first
        for (int pass = 0; pass < 2; ++pass) {
            a = 0; b = tv.cmp_dptr[c];
            while (a < tv.cmp_vlen || b < be) {
                const int32_t pv = a < tv.cmp_vlen ? tv.cmp_v[a] : 0x7fffffff;
                const int32_t pd = b < be ? tv.cmp_dpos[b] : 0x7fffffff;
                if (pv == pd) { ++a; ++b; continue; }
                const int64_t j = i + (pv < pd ? pv : pd);
                if (pv < pd) ++a; else ++b;
                if (pass == 0 && j >= n) row[have++] = (int32_t)(j - n);
                if (pass == 1 && j < n) row[have++] = (int32_t)j;
            }
        }
    }
}

static unsigned grid_for(int64_t items) {
    int64_t b = (items + 255) / 256;
    if (b < 1) b = 1;
    if (b > 148 * 32) b = 148 * 32;
    return (unsigned)b;
}

int32_t topo_build(net* h) {
    const net_topology& t = h->desc.topo;
    TopoView& tv = h->tv;
    memset(&tv, 0, sizeof(tv));
    tv.kind = t.kind;
    tv.ndim = t.ndim;
    tv.nx = tv.ny = tv.nz = 1;
    tv.P = t.radius;
    tv.include_self = t.include_self ? 1 : 0;
    tv.ring_n = h->n / (h->desc.batch > 0 ? h->desc.batch : 1);
    const int64_t rn = tv.ring_n, nb = h->desc.batch > 0 ? h->desc.batch : 1;     // elements of one replica, replicas
    cudaStream_t st = h->stream;
    OSC_CUDA(h, cudaMemsetAsync(h->b.flag, 0, 4 * sizeof(int32_t), st));
    if (t.kind == NET_TOPO_RING) {
        h->degree_uniform = 2 * t.radius + tv.include_self;
        h->nnz = h->n * (int64_t)h->degree_uniform;
    } else if (t.kind == NET_TOPO_LATTICE) {
        tv.nx = (int32_t)t.extent[0];
        tv.ny = t.ndim >= 2 ? (int32_t)t.extent[1] : 1;
        tv.nz = t.ndim >= 3 ? (int32_t)t.extent[2] : 1;
        tv.noff = topo_lattice_noff(t.ndim, t.radius, tv.include_self);
        tv.off = h->b.off;
        lattice_offsets_kernel<<<1, 256, 0, st>>>(t.ndim, t.radius, tv.include_self, h->b.off, h->b.flag + 3);
        h->launches += 1;
        OSC_CUDA(h, cudaGetLastError());
        int32_t cnt = -1;
        OSC_CUDA(h, cudaMemcpyAsync(&cnt, h->b.flag + 3, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        OSC_CUDA(h, cudaStreamSynchronize(st));
        if (cnt != tv.noff) return set_err(h, NET_ERR_TOPOLOGY, "lattice offset table: built %d entries, expected %d", cnt, tv.noff);
        h->degree_uniform = tv.noff;
        h->nnz = h->n * (int64_t)tv.noff;
    } else if (t.kind == NET_TOPO_CSR) {
        cudaMemcpyKind kind = t.ptrs_are_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        OSC_CUDA(h, cudaMemcpyAsync(h->b.row_ptr, t.row_ptr, sizeof(int64_t) * (rn + 1), kind, st));
        if (t.nnz > 0)
            OSC_CUDA(h, cudaMemcpyAsync(h->b.col_idx, t.col_idx, sizeof(int32_t) * t.nnz, kind, st));
        csr_validate_kernel<<<grid_for(t.nnz > rn ? t.nnz : rn), 256, 0, st>>>(h->b.row_ptr, h->b.col_idx, rn, t.nnz, h->b.flag);
        csr_degree_kernel<<<grid_for(rn), 256, 0, st>>>(h->b.row_ptr, rn, h->b.flag);
        h->launches += 2;
        OSC_CUDA(h, cudaGetLastError());
        int32_t f[4];
        OSC_CUDA(h, cudaMemcpyAsync(f, h->b.flag, sizeof(f), cudaMemcpyDeviceToHost, st));
        OSC_CUDA(h, cudaStreamSynchronize(st));
        if (f[0] & 1) return set_err(h, NET_ERR_TOPOLOGY, "CSR row_ptr is not monotone from 0 to nnz");
        if (f[0] & 2) return set_err(h, NET_ERR_TOPOLOGY, "CSR col_idx has an index outside [0, n)");
        tv.row_ptr = h->b.row_ptr;
        tv.col_idx = h->b.col_idx;
        h->nnz = t.nnz * nb;
        h->degree_uniform = f[2] ? -1 : f[1];
    } else if (t.kind == NET_TOPO_COMPRESSED) {
        // V, D, C of Alg. 2 go to the workspace as they are; validated on the host
        const net_compressed* c = t.compressed;
        const int64_t n = rn, dtot = c->d_ptr[c->k];
        for (int64_t q = 0; q < c->v_len; ++q)
            if (c->v_pos[q] < 0 || c->v_pos[q] >= n || (q > 0 && c->v_pos[q] <= c->v_pos[q - 1]))
                return set_err(h, NET_ERR_TOPOLOGY, "compressed matrix: common vector not sorted / out of range");
        int32_t* deg = (int32_t*)malloc(sizeof(int32_t) * (size_t)c->k);
        if (!deg) return set_err(h, NET_ERR_INVALID, "out of host memory");
        int32_t maxdeg = 0;
        for (int64_t e = 0; e < c->k; ++e) {
            const int64_t b = c->d_ptr[e], be = c->d_ptr[e + 1];
            if (be < b || be > dtot) { free(deg); return set_err(h, NET_ERR_TOPOLOGY, "compressed matrix: d_ptr not monotone"); }
            int64_t common = 0, a = 0;
            for (int64_t q = b; q < be; ++q) {
                const int32_t p = c->d_pos[q];
                if (p < 0 || p >= n || (q > b && p <= c->d_pos[q - 1])) { free(deg); return set_err(h, NET_ERR_TOPOLOGY, "compressed matrix: table entry not sorted / out of range"); }
                while (a < c->v_len && c->v_pos[a] < p) ++a;
                if (a < c->v_len && c->v_pos[a] == p) ++common;
            }
            deg[e] = (int32_t)(c->v_len + (be - b) - 2 * common);      // |V xor D_e|
            if (deg[e] > maxdeg) maxdeg = deg[e];
        }
        int64_t nnz = 0;
        bool uniform = true;
        for (int64_t i = 0; i < n; ++i) {
            if (c->c[i] < 0 || c->c[i] >= c->k) { free(deg); return set_err(h, NET_ERR_TOPOLOGY, "compressed matrix: row reference outside the table"); }
            nnz += deg[c->c[i]];
            uniform = uniform && deg[c->c[i]] == deg[c->c[0]];
        }
        OSC_CUDA(h, cudaMemcpyAsync(h->b.cmp_v, c->v_pos, sizeof(int32_t) * c->v_len, cudaMemcpyHostToDevice, st));
        OSC_CUDA(h, cudaMemcpyAsync(h->b.cmp_dptr, c->d_ptr, sizeof(int64_t) * (c->k + 1), cudaMemcpyHostToDevice, st));
        if (dtot > 0) OSC_CUDA(h, cudaMemcpyAsync(h->b.cmp_dpos, c->d_pos, sizeof(int32_t) * dtot, cudaMemcpyHostToDevice, st));
        OSC_CUDA(h, cudaMemcpyAsync(h->b.cmp_c, c->c, sizeof(int32_t) * n, cudaMemcpyHostToDevice, st));
        OSC_CUDA(h, cudaMemcpyAsync(h->b.cmp_deg, deg, sizeof(int32_t) * c->k, cudaMemcpyHostToDevice, st));
        OSC_CUDA(h, cudaStreamSynchronize(st));
        h->degree_uniform = uniform ? deg[c->c[0]] : -1;
        free(deg);
        tv.cmp_v = h->b.cmp_v; tv.cmp_dptr = h->b.cmp_dptr; tv.cmp_dpos = h->b.cmp_dpos;
        tv.cmp_c = h->b.cmp_c; tv.cmp_deg = h->b.cmp_deg;
        tv.cmp_vlen = (int32_t)c->v_len; tv.cmp_k = (int32_t)c->k; tv.cmp_maxdeg = maxdeg;
        h->nnz = nnz;
    } else {  // RANDOM_INDEGREE
        random_indegree_kernel<<<grid_for(rn), 256, 0, st>>>(rn, t.in_degree, t.seed, h->b.col_idx);
        uniform_row_ptr_kernel<<<grid_for(rn + 1), 256, 0, st>>>(h->b.row_ptr, rn, t.in_degree);
        h->launches += 2;
        OSC_CUDA(h, cudaGetLastError());
        tv.k_uniform = t.in_degree;
        tv.row_ptr = h->b.row_ptr;
        tv.col_idx = h->b.col_idx;
        h->nnz = h->n * (int64_t)t.in_degree;
        h->degree_uniform = t.in_degree;
    }
    return NET_OK;
}

int32_t topo_expand(net* h, int64_t row_begin, int64_t row_count, int64_t* d_row_ptr,
                    int32_t* d_col_idx) {
    cudaStream_t st = h->stream;
    if (h->tv.kind == NET_TOPO_COMPRESSED) {
        compressed_degree_kernel<<<grid_for(row_count + 1), 256, 0, st>>>(h->tv, row_begin, row_count, d_row_ptr);
        scan_i64_kernel<<<1, 1024, 0, st>>>(d_row_ptr, row_count);
        if (row_count > 0) compressed_expand_kernel<<<grid_for(row_count), 256, 0, st>>>(h->tv, h->n, row_begin, row_count, d_row_ptr, d_col_idx);
        h->launches += 3;
        OSC_CUDA(h, cudaGetLastError());
        return NET_OK;
    }
    if (h->tv.kind == NET_TOPO_RING || h->tv.kind == NET_TOPO_LATTICE) {
        int32_t deg = h->degree_uniform;
        uniform_row_ptr_kernel<<<grid_for(row_count + 1), 256, 0, st>>>(d_row_ptr, row_count, deg);
        if (row_count > 0 && deg > 0 && h->tv.kind == NET_TOPO_RING)
            expand_ring_kernel<<<grid_for(row_count * (int64_t)deg), 256, 0, st>>>(h->tv.ring_n, h->tv.P, h->tv.include_self, row_begin, row_count, deg, d_col_idx);
        else if (row_count > 0)
            expand_rows_kernel<<<grid_for(row_count), 256, 0, st>>>(h->tv, h->n, row_begin, row_count, deg, d_col_idx);
        h->launches += 2;
    } else {
        copy_rows_kernel<<<grid_for(row_count + 1), 256, 0, st>>>(h->b.row_ptr, h->b.col_idx, row_begin, row_count, d_row_ptr, d_col_idx, h->tv.ring_n);
        h->launches += 1;
    }
    OSC_CUDA(h, cudaGetLastError());
    return NET_OK;
}

}  // namespace oscnet
