// bsh_post.cuh -- post-processing of the toplists on the GPU: parameter-space distance, coincidences between
// two lists, clusters (connected components), significance-weighted centroids.
//
//   PAPER.md section V.E, L385-L407.  Distance, Eq. (44) L395 with "a mean of the resolution at both points" (L399):
//       d^2(a, b) = sum_k [ (p_k(a) - p_k(b)) / ((delta_k(a) + delta_k(b)) / 2) ]^2,   k = f, x, y, a_p, Omega, t_asc.
//   Every operation is one rounded FP64 operation in the order written, the squares added left to right (R-25),
//   so that the decisions d < window are the same on every implementation of this order.
//
// Lists are small (<= 5000 candidates per 0.1 Hz band, L496): the all-pairs adjacency is a bit matrix (one ballot per 32
// pairs), connected components are found by min-label propagation with pointer jumping on that matrix (a cluster's label
// is the smallest index of its members, which is unique), and the per-cluster sums run over the members in index order
// (deterministic FP64 sums).  None of this is on the hot path; it completes the pipeline of Fig. 4.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsh {

constexpr int kNPar = 6;

__device__ __forceinline__ double post_distance2(const double *__restrict__ pa, const double *__restrict__ ra,
                                                 const double *__restrict__ pb, const double *__restrict__ rb)
{
    double d2 = 0.0;
#pragma unroll
    for (int k = 0; k < kNPar; ++k) {
        const double res = __dmul_rn(0.5, __dadd_rn(ra[k], rb[k]));           // mean of the two resolutions, L399
        const double q = __ddiv_rn(__dsub_rn(pa[k], pb[k]), res);
        d2 = __dadd_rn(d2, __dmul_rn(q, q));                                  // Eq. (44)
    }
    return d2;
}

// adj[a][w] bit b = (d(a, 32 w + b) < window) for a in list A (rows), b in list B (columns); self pairs excluded when the
// two lists are the same array (same != 0).  One warp per (row, word).
__global__ void __launch_bounds__(256) post_adjacency_kernel(int na, const double *__restrict__ pa, const double *__restrict__ ra,
                                                             int nb, const double *__restrict__ pb, const double *__restrict__ rb,
                                                             double w2, int same, int words, uint32_t *__restrict__ adj,
                                                             int32_t *__restrict__ row_count)
{
    const int64_t gw = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (gw >= (int64_t)na * words) return;
    const int a = (int)(gw / words), w = (int)(gw % words);
    const int b = 32 * w + lane;
    bool on = false;
    if (b < nb && !(same && a == b)) on = post_distance2(pa + kNPar * (int64_t)a, ra + kNPar * (int64_t)a, pb + kNPar * (int64_t)b,
                                                         rb + kNPar * (int64_t)b) < w2;
    const uint32_t word = __ballot_sync(0xFFFFFFFFu, on);
    if (lane == 0) {
        adj[(int64_t)a * words + w] = word;
        if (row_count && word) atomicAdd(row_count + a, __popc(word));
    }
}

__global__ void post_iota_kernel(int n, int32_t *label)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) label[i] = i;
}

// one sweep of min-label propagation over the adjacency rows, followed by pointer jumping; *changed is set when any label
// moved.  Labels only ever decrease and always name a member of the same component, so stale reads are harmless.
__global__ void __launch_bounds__(256) post_propagate_kernel(int n, int words, const uint32_t *__restrict__ adj, int32_t *label,
                                                             int *changed)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int32_t m = label[i];
    const int32_t before = m;
    for (int w = 0; w < words; ++w) {
        uint32_t bits = adj[(int64_t)i * words + w];
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            const int32_t l = label[32 * w + b];
            m = l < m ? l : m;
        }
    }
    for (int32_t l = label[m]; l < m; l = label[m]) m = l;                    // pointer jumping
    if (m < before) {
        atomicMin(label + i, m);
        *changed = 1;
    }
}

// Option B (L403): per cluster the top template (largest significance, smallest index among equals) ...
__global__ void __launch_bounds__(256) post_top_kernel(int n, const int32_t *__restrict__ label, const double *__restrict__ sig,
                                                       int32_t *__restrict__ top)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    int32_t t = -1;
    if (label[c] == c)
        for (int m = 0; m < n; ++m)
            if (label[m] == c && (t < 0 || sig[m] > sig[t])) t = m;
    top[c] = t;
}

// ... and members at prune_window or further from it are removed (label -1)
__global__ void __launch_bounds__(256) post_prune_kernel(int n, const double *__restrict__ p, const double *__restrict__ r,
                                                         const int32_t *__restrict__ top, double pw2, int32_t *label)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const int32_t c = label[m];
    const int32_t t = top[c];
    const bool keep = m == t || post_distance2(p + kNPar * (int64_t)m, r + kNPar * (int64_t)m, p + kNPar * (int64_t)t,
                                               r + kNPar * (int64_t)t) < pw2;
    label[m] = keep ? c : -1;
}

// Step 3 (L405): per cluster (thread = candidate index that is a label) the significance-weighted centroid, the summed
// significance and the member count, members taken in index order.
__global__ void __launch_bounds__(128) post_centroid_kernel(int n, const double *__restrict__ p, const double *__restrict__ sig,
                                                            const int32_t *__restrict__ label, double *__restrict__ cen_by_label,
                                                            double *__restrict__ sig_by_label, int32_t *__restrict__ members_by_label)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    double acc[kNPar] = {0, 0, 0, 0, 0, 0}, ssum = 0.0;
    int32_t members = 0;
    for (int m = 0; m < n; ++m)
        if (label[m] == c) {
            members += 1;
            ssum = __dadd_rn(ssum, sig[m]);
#pragma unroll
            for (int k = 0; k < kNPar; ++k) acc[k] = __dadd_rn(acc[k], __dmul_rn(sig[m], p[kNPar * (int64_t)m + k]));
        }
    members_by_label[c] = members;
    sig_by_label[c] = ssum;
#pragma unroll
    for (int k = 0; k < kNPar; ++k) cen_by_label[kNPar * (int64_t)c + k] = members ? __ddiv_rn(acc[k], ssum) : 0.0;
}

// Compaction in increasing label order + the most significant cluster (first among equals).  One block.
__global__ void __launch_bounds__(1024) post_compact_kernel(int n, const double *__restrict__ cen_by_label,
                                                            const double *__restrict__ sig_by_label,
                                                            const int32_t *__restrict__ members_by_label, int32_t *__restrict__ root,
                                                            double *__restrict__ centroid, double *csig,
                                                            int32_t *__restrict__ n_members, int32_t *__restrict__ out2)
{
    __shared__ int s_base, s_warp[32];
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int c0 = 0; c0 < n; c0 += 1024) {
        const int c = c0 + threadIdx.x;
        const bool is = c < n && members_by_label[c] > 0;
        const uint32_t bal = __ballot_sync(0xFFFFFFFFu, is);
        if (lane == 0) s_warp[warp] = __popc(bal);
        __syncthreads();
        int off = s_base;
        for (int w = 0; w < warp; ++w) off += s_warp[w];
        if (is) {
            const int pos = off + __popc(bal & ((1u << lane) - 1u));
            root[pos] = c;
            n_members[pos] = members_by_label[c];
            csig[pos] = sig_by_label[c];
            for (int k = 0; k < kNPar; ++k) centroid[kNPar * (int64_t)pos + k] = cen_by_label[kNPar * (int64_t)c + k];
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
            for (int w = 0; w < 32; ++w) t += s_warp[w];
            s_base += t;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        int best = -1;
        for (int q = 0; q < s_base; ++q)
            if (best < 0 || csig[q] > csig[best]) best = q;
        out2[0] = s_base;
        out2[1] = best;
    }
}

// exclusive prefix sum of the row counts (one block), total in out[n]
__global__ void __launch_bounds__(1024) post_scan_kernel(int n, const int32_t *__restrict__ cnt, int64_t *__restrict__ off)
{
    __shared__ int64_t s_base;
    __shared__ int s_warp[32];
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i0 = 0; i0 < n; i0 += 1024) {
        const int i = i0 + threadIdx.x;
        int v = i < n ? cnt[i] : 0, x = v;
        for (int d = 1; d < 32; d <<= 1) {
            const int y = __shfl_up_sync(0xFFFFFFFFu, x, d);
            if (lane >= d) x += y;
        }
        if (lane == 31) s_warp[warp] = x;
        __syncthreads();
        int64_t o = s_base;
        for (int w = 0; w < warp; ++w) o += s_warp[w];
        if (i < n) off[i] = o + x - v;
        __syncthreads();
        if (threadIdx.x == 0) {
            int64_t t = 0;
            for (int w = 0; w < 32; ++w) t += s_warp[w];
            s_base += t;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) off[n] = s_base;
}

// Step 1 (L387-L393): the coincidental pairs in (a, b) order, their centroid "weighted by significance" and summed significance
__global__ void __launch_bounds__(256) post_pairs_kernel(int na, int words, const uint32_t *__restrict__ adj,
                                                         const int64_t *__restrict__ off, const double *__restrict__ pa,
                                                         const double *__restrict__ sa, const double *__restrict__ pb,
                                                         const double *__restrict__ sb, int64_t max_pairs,
                                                         int32_t *__restrict__ pair_a, int32_t *__restrict__ pair_b,
                                                         double *__restrict__ centroid, double *__restrict__ psig)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= na) return;
    int64_t pos = off[a];
    for (int w = 0; w < words; ++w) {
        uint32_t bits = adj[(int64_t)a * words + w];
        while (bits) {
            const int b = 32 * w + __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < max_pairs) {
                pair_a[pos] = a;
                pair_b[pos] = b;
                const double s = __dadd_rn(sa[a], sb[b]);
                psig[pos] = s;
#pragma unroll
                for (int k = 0; k < kNPar; ++k)
                    centroid[kNPar * pos + k] = __ddiv_rn(__dadd_rn(__dmul_rn(sa[a], pa[kNPar * (int64_t)a + k]),
                                                                    __dmul_rn(sb[b], pb[kNPar * (int64_t)b + k])), s);
            }
            pos += 1;
        }
    }
}

}  // namespace bsh
