// tree.cu -- step a0 (second half): implicit 32-ary tree over the sorted leaves and the leaf interaction list.
//
// "leaf metadata includes a baryon interaction domain, calculated by extending the bounding box to
// enclose the maximal smoothing length of the particles within the leaf ... all hydro operators utilize the same
// interaction list, which need only be assembled once per hydro subcycle, and reused for each kernel."
// Here the list of leaf a holds every leaf b whose periodic box-to-box gap is below max(hmax(a), hmax(b)); a flag
// marks the entries that also satisfy the one-sided criterion gap < hmax(a) used by the gather passes.
// The gap is evaluated with the same float operation sequence as the particle predicate (S3), so by
// monotonicity of IEEE rounding the list is an exact superset of the interacting particle pairs.
#include "crk_internal.cuh"

namespace {

struct Levels {
    int n_levels;
    int64_t off[CRK_MAX_LEVELS + 1];
    int64_t cnt[CRK_MAX_LEVELS + 1];
};

__global__ void __launch_bounds__(256) k_tree_level(float4* __restrict__ lo, float4* __restrict__ hi, int64_t in_off,
                                                    int64_t in_cnt, int64_t out_off, int64_t out_cnt) {
    const int lane = threadIdx.x & 31;
    const int64_t node = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (node >= out_cnt) return;
    const int64_t ch = node * CRK_BVH_FAN + lane;
    const float inf = __int_as_float(0x7f800000);
    float4 a = make_float4(inf, inf, inf, 0.f), b = make_float4(-inf, -inf, -inf, inf);
    if (ch < in_cnt) {
        a = lo[in_off + ch];
        b = hi[in_off + ch];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a.x = fminf(a.x, __shfl_xor_sync(0xffffffffu, a.x, o));
        a.y = fminf(a.y, __shfl_xor_sync(0xffffffffu, a.y, o));
        a.z = fminf(a.z, __shfl_xor_sync(0xffffffffu, a.z, o));
        a.w = fmaxf(a.w, __shfl_xor_sync(0xffffffffu, a.w, o));
        b.x = fmaxf(b.x, __shfl_xor_sync(0xffffffffu, b.x, o));
        b.y = fmaxf(b.y, __shfl_xor_sync(0xffffffffu, b.y, o));
        b.z = fmaxf(b.z, __shfl_xor_sync(0xffffffffu, b.z, o));
        b.w = fminf(b.w, __shfl_xor_sync(0xffffffffu, b.w, o));
    }
    if (lane == 0) {
        lo[out_off + node] = a;
        hi[out_off + node] = b;
    }
}

// lower bound of |wrap(x_i - x_j)| on one axis for x_i in [qlo,qhi], x_j in [blo,bhi]
__device__ __forceinline__ float axis_gap(float qlo, float qhi, float blo, float bhi, float L, float half, bool& wrap) {
    const float dmin = __fsub_rn(qlo, bhi);
    const float dmax = __fsub_rn(qhi, blo);
    wrap = wrap || (dmin < -half) || (dmax > half);
    const float g0 = fmaxf(0.f, fmaxf(dmin, -dmax));
    const float gp = fmaxf(0.f, fmaxf(__fsub_rn(L, dmax), __fsub_rn(dmin, L)));
    const float gm = fmaxf(0.f, fmaxf(__fadd_rn(dmin, L), __fsub_rn(-L, dmax)));
    return fminf(g0, fminf(gp, gm));
}

constexpr int NBR_WARPS = 8;
constexpr int NBR_STACK = 32 * (CRK_MAX_LEVELS + 1);

// One traversal per query leaf.  Leaf q owns slots [q * cap, (q + 1) * cap) of the list; entries beyond cap are counted but
// not written, and the host re-runs the kernel with a larger cap if the largest count (atomicMax -> *max_cnt) exceeds it
// (the capacity found is kept in the context, so later builds need one pass and no prefix sum).
// A level-1 node whose supports differ a lot (a background particle of large h among cluster particles) would hand the reach
// of its largest h to all 32 leaves in the joint traversal: its leaves take the per-leaf traversal instead (clustered 128^3:
// joint for all nodes 0.26 ms, per leaf 0.18 ms).
__device__ __forceinline__ bool node_is_mixed(float hmax, float hmin) { return hmax > 1.5f * hmin; }
// A set whose supports span more than a factor four (the Plummer configurations) is served leaf by leaf altogether: there the
// joint traversal loses even on the nodes of similar supports.  Decided once per build from the top level of the tree
// (k_set_mixed -> status word FW_SETMIXED).
__device__ __forceinline__ bool set_is_mixed(const float4* __restrict__ lo, const float4* __restrict__ hi, const Levels& lv, int lane) {
    const int top = lv.n_levels - 1;
    float hmax = 0.f, hmin = __int_as_float(0x7f800000);
    for (int64_t k = lane; k < lv.cnt[top]; k += 32) {
        hmax = fmaxf(hmax, lo[lv.off[top] + k].w);
        hmin = fminf(hmin, hi[lv.off[top] + k].w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        hmax = fmaxf(hmax, __shfl_xor_sync(0xffffffffu, hmax, o));
        hmin = fminf(hmin, __shfl_xor_sync(0xffffffffu, hmin, o));
    }
    return hmax > 4.0f * hmin;
}

__global__ void k_set_mixed(const float4* __restrict__ lo, const float4* __restrict__ hi, Levels lv, int* __restrict__ flag) {
    const bool mixed = set_is_mixed(lo, hi, lv, (int)threadIdx.x);
    if (threadIdx.x == 0) flag[FW_SETMIXED] = mixed ? 1 : 0;
}

// one traversal for query leaf q by the whole warp (stack = the warp's shared-memory stack)
__device__ __forceinline__ void leaf_list_one(const float4* __restrict__ lo, const float4* __restrict__ hi, const Levels& lv, float L,
                                              uint32_t cap, uint32_t* __restrict__ cnt, uint32_t* __restrict__ gcnt,
                                              uint32_t* __restrict__ list, uint32_t* __restrict__ max_cnt, uint32_t* stack_w,
                                              int64_t q, int lane) {
    const float4 qlo = lo[q], qhi = hi[q];
    const float hq2 = __fmul_rn(qlo.w, qlo.w);
    const float half = 0.5f * L;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t n_out = 0, n_gather = 0;
    const uint64_t base = (uint64_t)q * cap;
    int sp = 0;
    if (lane == 0) stack_w[0] = ((uint32_t)lv.n_levels << 28);   // pseudo-root: children = all nodes of the top level
    sp = 1;
    __syncwarp();
    while (sp > 0) {
        const uint32_t e = stack_w[sp - 1];
        --sp;
        __syncwarp();
        const int clev = (int)(e >> 28) - 1;
        const int64_t child = (int64_t)(e & CRK_LEAF_MASK) * CRK_BVH_FAN + lane;
        bool pass = false, gather = false, wrap = false;
        if (child < lv.cnt[clev]) {
            const float4 blo = lo[lv.off[clev] + child], bhi = hi[lv.off[clev] + child];
            const float gx = axis_gap(qlo.x, qhi.x, blo.x, bhi.x, L, half, wrap);
            const float gy = axis_gap(qlo.y, qhi.y, blo.y, bhi.y, L, half, wrap);
            const float gz = axis_gap(qlo.z, qhi.z, blo.z, bhi.z, L, half, wrap);
            const float g2 = __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
            const float hb2 = __fmul_rn(blo.w, blo.w);
            gather = g2 < hq2;
            pass = g2 < fmaxf(hq2, hb2);
        }
        const uint32_t m = __ballot_sync(0xffffffffu, pass);
        if (clev == 0) {
            const uint32_t mg = __ballot_sync(0xffffffffu, gather);
            if (pass) {
                const uint32_t pos = n_out + __popc(m & lt);
                if (pos < cap) list[base + pos] = (uint32_t)child | (gather ? CRK_FLAG_GATHER : 0u) | (wrap ? CRK_FLAG_WRAP : 0u);
            }
            n_out += __popc(m);
            n_gather += __popc(mg);
        } else {
            // push in descending order so that the lowest child is popped first (list comes out ascending)
            if (pass) stack_w[sp + __popc(m & ~lt & ~(1u << lane))] = ((uint32_t)clev << 28) | (uint32_t)child;
            sp += __popc(m);
            __syncwarp();
        }
    }
    if (lane == 0) {
        cnt[q] = n_out;
        gcnt[q] = n_gather;
        atomicMax(max_cnt, n_out);
    }
}

__global__ void __launch_bounds__(NBR_WARPS * 32) k_leaf_list(const float4* __restrict__ lo, const float4* __restrict__ hi,
                                                              Levels lv, float L, uint32_t cap, uint32_t* __restrict__ cnt,
                                                              uint32_t* __restrict__ gcnt, uint32_t* __restrict__ list,
                                                              uint32_t* __restrict__ max_cnt, const int* __restrict__ set_mixed) {
    __shared__ uint32_t stack[NBR_WARPS][NBR_STACK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t q = (int64_t)blockIdx.x * NBR_WARPS + w;
    if (q >= lv.cnt[0]) return;
    if (set_mixed && *set_mixed == 0) {   // the leaves of nodes with similar supports are served by k_leaf_list_joint
        const int64_t g = q / CRK_BVH_FAN;
        if (!node_is_mixed(lo[lv.off[1] + g].w, hi[lv.off[1] + g].w)) return;
    }
    leaf_list_one(lo, hi, lv, L, cap, cnt, gcnt, list, max_cnt, stack[w], q, lane);
}

// The same lists, built for the 32 leaves of a level-1 node together: one warp walks the tree ONCE with the node's box and
// largest h (a superset of what any of its leaves can reach: a leaf's box lies inside the node's, and the gap is evaluated
// with monotone float operations), collects the candidate leaves in ascending order in shared memory, and then every lane
// tests the candidates against its own leaf with exactly the arithmetic of k_leaf_list -- same entries, same order, a seventh
// of the instructions (the upper levels are pruned once per 32 leaves instead of once per leaf).
constexpr int JOINT_CHUNK = 128;
__global__ void __launch_bounds__(NBR_WARPS * 32) k_leaf_list_joint(const float4* __restrict__ lo, const float4* __restrict__ hi,
                                                                    Levels lv, float L, uint32_t cap, uint32_t* __restrict__ cnt,
                                                                    uint32_t* __restrict__ gcnt, uint32_t* __restrict__ list,
                                                                    uint32_t* __restrict__ max_cnt, const int* __restrict__ set_mixed) {
    __shared__ uint32_t stack[NBR_WARPS][NBR_STACK];
    __shared__ uint32_t chunk[NBR_WARPS][JOINT_CHUNK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t g = (int64_t)blockIdx.x * NBR_WARPS + w;          // level-1 node = leaves 32 g .. 32 g + 31
    if (g >= lv.cnt[1]) return;
    const float4 Qlo = lo[lv.off[1] + g], Qhi = hi[lv.off[1] + g];
    if (node_is_mixed(Qlo.w, Qhi.w) || *set_mixed != 0) return;     // served leaf by leaf (k_leaf_list)
    const float hQ2 = __fmul_rn(Qlo.w, Qlo.w);
    const int64_t q = g * CRK_BVH_FAN + lane;
    const bool valid = q < lv.cnt[0];
    const float inf = __int_as_float(0x7f800000);
    float4 qlo = make_float4(inf, inf, inf, 0.f), qhi = make_float4(-inf, -inf, -inf, 0.f);
    if (valid) {
        qlo = lo[q];
        qhi = hi[q];
    }
    const float hq2 = __fmul_rn(qlo.w, qlo.w);
    const float half = 0.5f * L;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t n_out = 0, n_gather = 0;
    const uint64_t base = (uint64_t)q * cap;
    int fill = 0;
    // every lane tests the collected candidate leaves against its own leaf (the arithmetic of k_leaf_list)
    auto drain = [&]() {
        __syncwarp();
        for (int t = 0; t < fill; ++t) {
            const uint32_t b = chunk[w][t];
            const float4 blo = lo[b], bhi = hi[b];
            bool wrap = false;
            const float gx = axis_gap(qlo.x, qhi.x, blo.x, bhi.x, L, half, wrap);
            const float gy = axis_gap(qlo.y, qhi.y, blo.y, bhi.y, L, half, wrap);
            const float gz = axis_gap(qlo.z, qhi.z, blo.z, bhi.z, L, half, wrap);
            const float g2 = __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
            const float hb2 = __fmul_rn(blo.w, blo.w);
            const bool gather = g2 < hq2;
            const bool pass = valid && (g2 < fmaxf(hq2, hb2));
            if (pass) {
                if (n_out < cap) list[base + n_out] = b | (gather ? CRK_FLAG_GATHER : 0u) | (wrap ? CRK_FLAG_WRAP : 0u);
                ++n_out;
                n_gather += gather ? 1u : 0u;
            }
        }
        fill = 0;
        __syncwarp();
    };
    int sp = 0;
    if (lane == 0) stack[w][0] = ((uint32_t)lv.n_levels << 28);   // pseudo-root: children = all nodes of the top level
    sp = 1;
    __syncwarp();
    while (sp > 0) {
        const uint32_t e = stack[w][sp - 1];
        --sp;
        __syncwarp();
        const int clev = (int)(e >> 28) - 1;
        const int64_t child = (int64_t)(e & CRK_LEAF_MASK) * CRK_BVH_FAN + lane;
        bool pass = false, wrap = false;
        if (child < lv.cnt[clev]) {
            const float4 blo = lo[lv.off[clev] + child], bhi = hi[lv.off[clev] + child];
            const float gx = axis_gap(Qlo.x, Qhi.x, blo.x, bhi.x, L, half, wrap);
            const float gy = axis_gap(Qlo.y, Qhi.y, blo.y, bhi.y, L, half, wrap);
            const float gz = axis_gap(Qlo.z, Qhi.z, blo.z, bhi.z, L, half, wrap);
            const float g2 = __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
            const float hb2 = __fmul_rn(blo.w, blo.w);
            pass = g2 < fmaxf(hQ2, hb2);
        }
        const uint32_t m = __ballot_sync(0xffffffffu, pass);
        if (clev == 0) {
            const int np = __popc(m);
            if (fill + np > JOINT_CHUNK) drain();
            if (pass) chunk[w][fill + __popc(m & lt)] = (uint32_t)child;
            fill += np;
        } else {
            // push in descending order so that the lowest child is popped first (candidates come out ascending)
            if (pass) stack[w][sp + __popc(m & ~lt & ~(1u << lane))] = ((uint32_t)clev << 28) | (uint32_t)child;
            sp += __popc(m);
            __syncwarp();
        }
    }
    drain();
    if (valid) {
        cnt[q] = n_out;
        gcnt[q] = n_gather;
    }
    const uint32_t mx = __reduce_max_sync(0xffffffffu, n_out);
    if (lane == 0) atomicMax(max_cnt, mx);
}

__global__ void k_sum_u32(const uint32_t* __restrict__ a, int64_t n, unsigned long long* __restrict__ out) {
    unsigned long long s = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) s += a[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(out, s);
}

}  // namespace

int crk_build_tree_and_list(crk_ctx* c) {
    float4* lo = (float4*)c->leaf_lo.p;
    float4* hi = (float4*)c->leaf_hi.p;
    Levels lv;
    lv.n_levels = c->n_levels;
    for (int l = 0; l <= CRK_MAX_LEVELS; ++l) {
        lv.off[l] = l < c->n_levels ? c->level_off[l] : 0;
        lv.cnt[l] = l < c->n_levels ? c->level_cnt[l] : 0;
    }
    for (int l = 1; l < c->n_levels; ++l) {
        const int wpb = 8;
        k_tree_level<<<(unsigned)((lv.cnt[l] + wpb - 1) / wpb), wpb * 32, 0, c->stream>>>(lo, hi, lv.off[l - 1],
                                                                                          lv.cnt[l - 1], lv.off[l],
                                                                                          lv.cnt[l]);
        CRK_TRY(crk_check_launch(c, "k_tree_level"));
    }
    const int64_t nl = c->nl;
    CRK_TRY(crk_ensure(c, c->nbr_cnt, (size_t)(nl + 1) * sizeof(uint32_t)));
    CRK_TRY(crk_ensure(c, c->nbr_gcnt, (size_t)(nl + 1) * sizeof(uint32_t)));
    const unsigned grid = (unsigned)((nl + NBR_WARPS - 1) / NBR_WARPS);
    // Leaf q owns a fixed slice of leaf_list_cap entries; the largest count and the pair totals go to the status words and are
    // checked by crk_build_cells at its single synchronisation (a list that overflowed its slice is rebuilt with a larger cap)
    uint32_t* d_max = (uint32_t*)c->flag.p + FW_MAXLIST;
    unsigned long long* d_sum = (unsigned long long*)((int*)c->flag.p + FW_SUM_GATHER);
    unsigned long long* d_sum2 = (unsigned long long*)((int*)c->flag.p + FW_SUM_ALL);
    if (c->leaf_list_cap < 64) c->leaf_list_cap = 96;
    CRK_TRY(crk_ensure(c, c->nbr_list, ((size_t)nl * c->leaf_list_cap + 1) * sizeof(uint32_t)));
    // enough level-1 nodes to fill the GPU with one warp each: the joint traversal for nodes of similar supports, the
    // per-leaf traversal for the rest; small sets: per leaf only
    const bool joint = c->n_levels >= 2 && lv.cnt[1] >= 2048 && !(c->prm.flags & CRK_FLAG_TREE_PER_LEAF);
    const int* d_mixed = (const int*)c->flag.p + FW_SETMIXED;
    if (joint) {
        k_set_mixed<<<1, 32, 0, c->stream>>>(lo, hi, lv, (int*)c->flag.p);
        CRK_TRY(crk_check_launch(c, "k_set_mixed"));
        const unsigned jgrid = (unsigned)((lv.cnt[1] + NBR_WARPS - 1) / NBR_WARPS);
        k_leaf_list_joint<<<jgrid, NBR_WARPS * 32, 0, c->stream>>>(lo, hi, lv, c->prm.box, (uint32_t)c->leaf_list_cap,
                                                                   (uint32_t*)c->nbr_cnt.p, (uint32_t*)c->nbr_gcnt.p,
                                                                   (uint32_t*)c->nbr_list.p, d_max, d_mixed);
        CRK_TRY(crk_check_launch(c, "k_leaf_list_joint"));
    }
    k_leaf_list<<<grid, NBR_WARPS * 32, 0, c->stream>>>(lo, hi, lv, c->prm.box, (uint32_t)c->leaf_list_cap,
                                                        (uint32_t*)c->nbr_cnt.p, (uint32_t*)c->nbr_gcnt.p,
                                                        (uint32_t*)c->nbr_list.p, d_max, joint ? d_mixed : nullptr);
    CRK_TRY(crk_check_launch(c, "k_leaf_list"));
    k_sum_u32<<<148, 256, 0, c->stream>>>((const uint32_t*)c->nbr_gcnt.p, nl, d_sum);
    CRK_TRY(crk_check_launch(c, "k_sum_u32"));
    k_sum_u32<<<148, 256, 0, c->stream>>>((const uint32_t*)c->nbr_cnt.p, nl, d_sum2);
    return crk_check_launch(c, "k_sum_u32");
}
