// frost_split.cu -- spatial splitting of a fast hierarchy level (the paper names the
// idea only; the definition is DESIGN.md reading 24): the fast set F of an entry is cut
// into the connected components of its fast pairs (symmetrised pair step below tau_pivot, Eq. 49-54),
// each component recurses on its own, and the slow pairs between components join the inter-level
// kick.  The time-step sweep of the entry has united the fast pairs in a union-find forest over the
// list positions of the entry's set (TimestepEdgePolicy / SymTimestepEdge); this file turns the
// forest into
//   * a label per list position (-1 = slow) for the masked kick sweeps,
//   * F reordered so that every component is contiguous (components by their smallest member,
//     members ascending -- a stable radix sort by label), and
//   * descriptor lists {offset, size} of the components by size class, on the device, so that all
//     small components of the entry are advanced by ONE batched launch (frost_small.cu).
#include <cub/cub.cuh>

#include "frost_common.cuh"

namespace frost {

__global__ void split_label_kernel(const int *__restrict__ forest, const double *__restrict__ tau,
                                   const int32_t *__restrict__ set, int n_set, double pivot,
                                   int *__restrict__ labpos, int *__restrict__ labg) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_set) return;
    const int g = set ? set[k] : k;
    const int l = (tau[g] >= pivot) ? -1 : uf_find(forest, k);
    labpos[k] = l;
    labg[g] = l;
}

__global__ void split_keys_kernel(const int32_t *__restrict__ F, int nF, const int *__restrict__ labg,
                                  int *__restrict__ keys) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < nF) keys[p] = labg[F[p]];
}

// hdr: [0] components, [1] small, [2] medium, [3] big, [4..5] sum of squared sizes (64 bit)
__global__ void split_classify_kernel(const int *__restrict__ sizes, const int *__restrict__ offs,
                                      const int *__restrict__ n_runs, int warp_max, int small_max,
                                      int2 *__restrict__ d_small, int2 *__restrict__ d_med,
                                      int2 *__restrict__ d_big, int big_cap, int *__restrict__ hdr) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = *n_runs;
    if (r == 0) hdr[0] = m;
    if (r >= m) return;
    const int sz = sizes[r], off = offs[r];
    atomicAdd((unsigned long long *)(hdr + 4), (unsigned long long)sz * (unsigned long long)sz);
    if (sz <= warp_max) d_small[atomicAdd(&hdr[1], 1)] = make_int2(off, sz);
    else if (sz <= small_max) d_med[atomicAdd(&hdr[2], 1)] = make_int2(off, sz);
    else {
        const int q = atomicAdd(&hdr[3], 1);
        if (q < big_cap) d_big[q] = make_int2(off, sz);
    }
}

static size_t align256(size_t v) { return (v + 255) / 256 * 256; }

int split_components(frost_ctx *c, int level, int ld, const double *tau, const int32_t *set, int n_set,
                     double pivot, const int *forest, const int32_t *F, int nF, SplitInfo *out) {
    *out = SplitInfo{};
    if (nF <= 0) return FROST_OK;
    constexpr int kBigCap = 64;
    // persistent part (lives as long as the entry): C, labpos, descriptors, header
    const size_t oC = 0, oLab = align256(oC + (size_t)nF * 4), oDs = align256(oLab + (size_t)n_set * 4);
    const size_t oDm = align256(oDs + (size_t)(nF / 2 + 1) * 8), oDb = align256(oDm + (size_t)(nF / 2 + 1) * 8);
    const size_t oHdr = align256(oDb + (size_t)kBigCap * 8), oR = oHdr + 256;
    const size_t oLR = align256(oR + (size_t)nF * 4), persist = align256(oLR + (size_t)nF * 4);
    FROST_TRY(ensure(c, c->lvlC[level], persist));
    char *pb = (char *)c->lvlC[level].p;
    int32_t *C = (int32_t *)(pb + oC);
    int *labpos = (int *)(pb + oLab);
    int2 *d_small = (int2 *)(pb + oDs), *d_med = (int2 *)(pb + oDm), *d_big = (int2 *)(pb + oDb);
    int *hdr = (int *)(pb + oHdr);
    int32_t *Rl = (int32_t *)(pb + oR);
    int *labR = (int *)(pb + oLR);
    // transient part: global-indexed labels, keys, run-length encoding, cub scratch
    size_t t_sort = 0, t_rle = 0, t_scan = 0;
    int *nul = nullptr;
    int bits = 1;
    while ((1 << bits) < n_set) ++bits;
    cub::DeviceRadixSort::SortPairs(nullptr, t_sort, nul, nul, nul, nul, nF, 0, bits, c->stream);
    cub::DeviceRunLengthEncode::Encode(nullptr, t_rle, nul, nul, nul, nul, nF, c->stream);
    cub::DeviceScan::ExclusiveSum(nullptr, t_scan, nul, nul, nF, c->stream);
    size_t t_cub = t_sort > t_rle ? t_sort : t_rle;
    if (t_scan > t_cub) t_cub = t_scan;
    const size_t oG = 0, oK = align256(oG + (size_t)ld * 4), oKs = align256(oK + (size_t)nF * 4);
    const size_t oU = align256(oKs + (size_t)nF * 4), oSz = align256(oU + (size_t)nF * 4);
    const size_t oOf = align256(oSz + (size_t)nF * 4), oNr = align256(oOf + (size_t)nF * 4);
    const size_t oT = align256(oNr + 256), transient = oT + t_cub + 256;
    FROST_TRY(ensure(c, c->comp, transient));
    char *tb = (char *)c->comp.p;
    int *labg = (int *)(tb + oG), *keys = (int *)(tb + oK), *keys_s = (int *)(tb + oKs);
    int *uniq = (int *)(tb + oU), *sizes = (int *)(tb + oSz), *offs = (int *)(tb + oOf), *n_runs = (int *)(tb + oNr);
    void *tmp = tb + oT;

    split_label_kernel<<<(n_set + 255) / 256, 256, 0, c->stream>>>(forest, tau, set, n_set, pivot, labpos, labg);
    FROST_TRY(check_launch(c));
    split_keys_kernel<<<(nF + 255) / 256, 256, 0, c->stream>>>(F, nF, labg, keys);
    FROST_TRY(check_launch(c));
    FROST_CUDA(c, cub::DeviceRadixSort::SortPairs(tmp, t_cub, keys, keys_s, F, C, nF, 0, bits, c->stream));
    c->launches += 2;
    // (the scan below runs over nF entries of `sizes`, the encoder writes only the first *n_runs)
    FROST_CUDA(c, cudaMemsetAsync(sizes, 0, (size_t)nF * sizeof(int), c->stream));
    FROST_CUDA(c, cub::DeviceRunLengthEncode::Encode(tmp, t_cub, keys_s, uniq, sizes, n_runs, nF, c->stream));
    c->launches += 2;
    FROST_CUDA(c, cub::DeviceScan::ExclusiveSum(tmp, t_cub, sizes, offs, nF, c->stream));
    c->launches += 2;
    FROST_CUDA(c, cudaMemsetAsync(hdr, 0, 8 * sizeof(int), c->stream));
    split_classify_kernel<<<(nF + 255) / 256, 256, 0, c->stream>>>(sizes, offs, n_runs, comp_warp_max(), small_max(),
                                                                 d_small, d_med, d_big, kBigCap, hdr);
    FROST_TRY(check_launch(c));
    int h[8];
    FROST_CUDA(c, cudaMemcpyAsync(h, hdr, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    FROST_CUDA(c, cudaStreamSynchronize(c->stream));
    out->m = h[0]; out->n_small = h[1]; out->n_med = h[2]; out->n_big = h[3];
    unsigned long long ss;
    memcpy(&ss, h + 4, sizeof(ss));
    out->sumsq = (long long)ss;
    if (out->n_big > kBigCap) return FROST_ELIMIT;       // more than 64 components above 1024 particles
    if (out->n_big > 0) {
        int2 big[kBigCap];
        FROST_CUDA(c, cudaMemcpyAsync(big, d_big, (size_t)out->n_big * sizeof(int2), cudaMemcpyDeviceToHost, c->stream));
        FROST_CUDA(c, cudaStreamSynchronize(c->stream));
        // the append order of the classification kernel is arbitrary: sort by offset (components are
        // independent, but a fixed order keeps the launch sequence reproducible)
        for (int a = 0; a < out->n_big; ++a)
            for (int b = a + 1; b < out->n_big; ++b)
                if (big[b].x < big[a].x) { const int2 t = big[a]; big[a] = big[b]; big[b] = t; }
        for (int a = 0; a < out->n_big; ++a) { out->big_off[a] = big[a].x; out->big_size[a] = big[a].y; }
    }
    // kick decomposition (frost_api.cu: cross_kick): G = the largest component above 1024 particles, if
    // any; R = every other fast particle as one list with its labels (the sorted keys)
    int gb = -1;
    for (int a = 0; a < out->n_big; ++a)
        if (gb < 0 || out->big_size[a] > out->big_size[gb]) gb = a;
    if (gb >= 0) { out->g_off = out->big_off[gb]; out->g_size = out->big_size[gb]; }
    const int head = out->g_off, tail = nF - out->g_off - out->g_size;
    out->nR = head + tail;
    if (head > 0) {
        FROST_CUDA(c, cudaMemcpyAsync(Rl, C, (size_t)head * 4, cudaMemcpyDeviceToDevice, c->stream));
        FROST_CUDA(c, cudaMemcpyAsync(labR, keys_s, (size_t)head * 4, cudaMemcpyDeviceToDevice, c->stream));
    }
    if (tail > 0) {
        FROST_CUDA(c, cudaMemcpyAsync(Rl + head, C + out->g_off + out->g_size, (size_t)tail * 4,
                                      cudaMemcpyDeviceToDevice, c->stream));
        FROST_CUDA(c, cudaMemcpyAsync(labR + head, keys_s + out->g_off + out->g_size, (size_t)tail * 4,
                                      cudaMemcpyDeviceToDevice, c->stream));
    }
    out->R = Rl; out->labR = labR;
    out->C = C; out->labpos = labpos; out->desc_small = d_small; out->desc_med = d_med;
    out->n_small_dev = hdr + 1; out->n_med_dev = hdr + 2;
    return FROST_OK;
}

}  // namespace frost
