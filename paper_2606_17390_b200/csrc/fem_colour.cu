// Element colouring for atomics-free in-place assembly (assembly_mode 1).
// Two elements that share a node get different colours; fem_assemble then runs the element kernel colour by colour and
// adds K^e / R^e straight into csr_vals / residual with plain read-modify-write — no two elements of one launch touch
// the same entry, and the colour order fixes the summation order (deterministic; replaces unordered atomics and the
// triplet sort/merge of PAPER.md Alg. E1 :1037-1047).  The first contributor of every CSR block (in colour order) is
// marked at setup so that it stores instead of adding: outputs need no zero-fill.
// Colouring: Jones–Plassmann rounds with hashed priorities (deterministic: depends on element ids only).
#include "fem_internal.h"
#include <cub/device/device_radix_sort.cuh>
#include <stdio.h>

__device__ __forceinline__ unsigned int prio_hash(unsigned int e) {
    unsigned int x = e * 0x9E3779B1u;
    x ^= x >> 16; x *= 0x85EBCA6Bu; x ^= x >> 13; x *= 0xC2B2AE35u; x ^= x >> 16;
    return x;
}
// strict total order on elements: (hash, id)
__device__ __forceinline__ bool prio_greater(unsigned int a, unsigned int b) {
    const unsigned int ha = prio_hash(a), hb = prio_hash(b);
    return ha > hb || (ha == hb && a > b);
}

// One round: an uncoloured element whose priority beats all its uncoloured neighbours takes the smallest colour not used
// by its coloured neighbours.  colour_in is the state before the round (so the round is order-independent).
__global__ void k_colour_round(long long n_elems, const int *__restrict__ conn, const int *__restrict__ inc_ptr,
                               const int *__restrict__ inc, const signed char *__restrict__ colour_in,
                               signed char *__restrict__ colour_out, int *n_left, int *overflow) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n_elems) return;
    if (colour_in[e] >= 0) { colour_out[e] = colour_in[e]; return; }
    unsigned long long used = 0;
    bool wait = false;
    for (int a = 0; a < 8 && !wait; a++) {
        const int nd = conn[e * 8 + a];
        for (int j = inc_ptr[nd]; j < inc_ptr[nd + 1]; j++) {
            const int f = inc[j] >> 3;
            if (f == e) continue;
            const int cf = colour_in[f];
            if (cf >= 0) used |= 1ull << cf;
            else if (prio_greater((unsigned)f, (unsigned)e)) { wait = true; break; }
        }
    }
    if (wait) { colour_out[e] = -1; atomicAdd(n_left, 1); return; }
    const int c = __ffsll((long long)~used) - 1;
    if (c < 0 || c >= 63) { atomicOr(overflow, 1); colour_out[e] = 62; return; }
    colour_out[e] = (signed char)c;
}

__global__ void k_colour_keys(long long n_elems, const signed char *__restrict__ colour, unsigned char *keys, int *ids,
                              int *count /*[64]*/) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n_elems) return;
    keys[e] = (unsigned char)colour[e];
    ids[e] = (int)e;
    atomicAdd(&count[colour[e]], 1);
}

// First contributor (smallest (colour, element id)) of every node-pair block and of every node's residual.
// One thread per node; first_mask[e] bit (I*8+K) <=> element e stores (instead of adds) its block (I,K);
// first_res[e] bit I likewise for the residual of local node I.
__global__ void k_first_masks(long long n_nodes, const int *__restrict__ inc_ptr, const int *__restrict__ inc,
                              const int *__restrict__ nb_ptr, const unsigned char *__restrict__ elem_pos,
                              const signed char *__restrict__ colour, unsigned long long *first_mask,
                              unsigned int *first_res) {
    const long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    const int b = inc_ptr[n], m = inc_ptr[n + 1] - b, len = nb_ptr[n + 1] - nb_ptr[n];
    unsigned long long best[8 * FEM_MAX_NODE_ELEMS];   // per neighbour position: min key = colour<<40 | e<<8 | I*8+K... kept as (colour<<32 | e)
    for (int p = 0; p < len; p++) best[p] = ~0ull;
    unsigned long long rbest = ~0ull;
    int rarg = -1;
    for (int s = 0; s < m; s++) {
        const int t = inc[b + s], e = t >> 3;
        const unsigned long long key = ((unsigned long long)(unsigned char)colour[e] << 32) | (unsigned int)e;
        if (key < rbest) { rbest = key; rarg = t; }
        for (int K = 0; K < 8; K++) {
            const int p = elem_pos[(long long)t * 8 + K];
            if (key < best[p]) best[p] = key;
        }
    }
    // a collapsed element (same node twice) would own a block through two (I,K) pairs: only the first pair may store
    for (int s = 0; s < m; s++) {
        const int t = inc[b + s], e = t >> 3, I = t & 7;
        const unsigned long long key = ((unsigned long long)(unsigned char)colour[e] << 32) | (unsigned int)e;
        for (int K = 0; K < 8; K++) {
            const int p = elem_pos[(long long)t * 8 + K];
            if (best[p] == key) {
                atomicOr(&first_mask[e], 1ull << (I * 8 + K));
                best[p] = ~0ull - 1;   // taken
            }
        }
    }
    if (rarg >= 0) atomicOr(&first_res[rarg >> 3], 1u << (rarg & 7));
}

static inline unsigned cblk(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// Builds colour lists and first-writer masks.  Requires the pattern arrays.  Synchronises.
int fem_build_colouring(fem_ctx *c) {
    const long long ne = c->n_elems, nn = c->n_nodes;
    signed char *col[2] = {nullptr, nullptr};
    unsigned char *keys = nullptr, *keys_out = nullptr;
    int *ids = nullptr, *d_cnt = nullptr;
    void *tmp = nullptr;
    size_t tmp_bytes = 0;
    int rc = FEM_OK;
    do {
#define TRY(call) { cudaError_t _e = (call); if (_e != cudaSuccess) { rc = fem_cuda_fail(_e, #call); break; } }
        TRY(cudaMalloc(&col[0], ne));
        TRY(cudaMalloc(&col[1], ne));
        TRY(cudaMalloc(&d_cnt, sizeof(int) * 66));
        TRY(cudaMemset(col[0], 0xff, ne));
        int cur = 0, left = 1, rounds = 0, ovf = 0;
        while (left > 0 && rounds < 1000) {
            TRY(cudaMemset(d_cnt, 0, sizeof(int) * 2));
            k_colour_round<<<cblk(ne, 128), 128>>>(ne, c->d_conn, c->d_inc_ptr, c->d_inc, col[cur], col[cur ^ 1], d_cnt, d_cnt + 1);
            int h[2];
            TRY(cudaMemcpy(h, d_cnt, sizeof(h), cudaMemcpyDeviceToHost));
            left = h[0]; ovf |= h[1];
            cur ^= 1; rounds++;
        }
        if (rc != FEM_OK) break;
        if (left > 0 || ovf) { rc = FEM_ERR_DEGREE; break; }
        // elements grouped by colour, ascending id within a colour (stable radix sort on the colour byte)
        TRY(cudaMalloc(&keys, ne));
        TRY(cudaMalloc(&keys_out, ne));
        TRY(cudaMalloc(&ids, sizeof(int) * ne));
        TRY(cudaMalloc(&c->d_elist, sizeof(int) * ne));
        TRY(cudaMemset(d_cnt, 0, sizeof(int) * 66));
        k_colour_keys<<<cblk(ne, 256), 256>>>(ne, col[cur], keys, ids, d_cnt);
        TRY(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys_out, ids, c->d_elist, (int)ne, 0, 6));
        TRY(cudaMalloc(&tmp, tmp_bytes));
        TRY(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys_out, ids, c->d_elist, (int)ne, 0, 6));
        int hc[64];
        TRY(cudaMemcpy(hc, d_cnt, sizeof(hc), cudaMemcpyDeviceToHost));
        c->n_colours = 0;
        c->colour_start[0] = 0;
        for (int k = 0; k < 64; k++) {
            if (hc[k] == 0) break;
            c->colour_start[k + 1] = c->colour_start[k] + hc[k];
            c->n_colours = k + 1;
        }
        if (c->colour_start[c->n_colours] != ne) { rc = FEM_ERR_ARG; break; }
        TRY(cudaMalloc(&c->d_first_mask, sizeof(unsigned long long) * ne));
        TRY(cudaMalloc(&c->d_first_res, sizeof(unsigned int) * ne));
        TRY(cudaMemset(c->d_first_mask, 0, sizeof(unsigned long long) * ne));
        TRY(cudaMemset(c->d_first_res, 0, sizeof(unsigned int) * ne));
        k_first_masks<<<cblk(nn, 64), 64>>>(nn, c->d_inc_ptr, c->d_inc, c->d_nb_ptr, c->d_elem_pos, col[cur], c->d_first_mask,
                                            c->d_first_res);
        TRY(cudaGetLastError());
        TRY(cudaDeviceSynchronize());
        c->colour_rounds = rounds;
#undef TRY
    } while (0);
    void *fr[] = {col[0], col[1], keys, keys_out, ids, d_cnt, tmp};
    for (void *p : fr) if (p) cudaFree(p);
    return rc;
}
