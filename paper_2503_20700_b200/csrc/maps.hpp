// Tables handed to the device block-map builder (heff_maps.cu) and its entry point.  See heff_maps.cu.
#pragma once
#include <cuda_runtime_api.h>

#include <cstdint>
#include <vector>

#include "kernels.hpp"

namespace dmrg {

struct MapBlock { int l, ab, r, rows, cols, pad; int64_t off, poff; };       // one psi block (exchange layout + padded copy)
struct MapTerm { int opL, opR, dm, pd, pr, pad; double coef; };               // opL / opR: index into opsL / opsR or -1
struct MapOp { const double* base; int cls, trans, ref, pad; };               // (stored operator, transposed?) ; ref: stored operator id
struct MapSide {                                                               // quantum-number maps of one block's operator classes
    const int* out;       // [ncls * nsec] in-sector -> out-sector or -1
    const int* inv;       // [ncls * nsec] out-sector -> in-sector or -1
    const int64_t* off;   // [ncls * nsec] storage offset of the dense block of in-sector
    const int* dim;       // [nsec] sector dimensions
    int nsec, pad;
};
struct MapCtx {
    const MapBlock* blocks; const int* lookup;        // psi blocks, [nL * 16] -> block or -1
    const MapTerm* terms; const double* dm;            // terms, dot matrices [ndm][16][16] (row: output state)
    const MapOp* opsL; const MapOp* opsR;
    const int* refclsL; const int* refclsR;            // class of every stored operator id
    const int* nL; const int* dotqn;                   // particle number of the left sectors / of the 16 dot states
    MapSide L, R;
    int nblk, nterm, nopsL, nopsR, nrefL, nrefR;
    const double* xpad; double* y;                     // padded x and the output vector
};

struct MapChunkOut {                                  // device-resident launch descriptors of one chunk
    Task* tasks1 = nullptr; Seg* segs1 = nullptr; Tile* tiles1 = nullptr; int ntasks1 = 0, nsegs1 = 0, ntiles1 = 0;
    Task* tasks2 = nullptr; Seg* segs2 = nullptr; Tile* tiles2 = nullptr; int ntasks2 = 0, nsegs2 = 0, ntiles2 = 0;
    double flops1 = 0, flops2 = 0;
    int64_t t_doubles = 0;                            // intermediate buffer the chunk needs
    int split = 1;                                    // split-K parts of phase 2 actually used
};

// Scratch + results of the builder.  All device allocations go through alloc / are owned by the caller afterwards.
struct MapBuild {
    std::vector<int> chunk_begin;                     // term ranges [chunk_begin[c], chunk_begin[c+1])
    std::vector<MapChunkOut> chunks;
    DiagItemK* diag_items = nullptr; int* diag_ptr = nullptr; int ndiag = 0;
    double f_alg = 0, ngemm = 0, b_ops = 0;
};

// Phase A: usage / accounting pass over all terms; fills usage_host[nterm] (doubles of T each term needs), the stats and
// the diagonal items.  Phase B (per chunk, after the host has cut the term list into chunks and allocated T):
// emits tasks / segments / tiles.  dev_alloc_fn allocates device memory that the caller owns.
typedef void* (*MapAlloc)(size_t bytes);
void maps_usage(const MapCtx& cx, std::vector<double>& usage_host, MapBuild& out, MapAlloc alloc, void (*dealloc)(void*),
                cudaStream_t st);
// S: split-K parts of phase 2 (part 0 -> y, parts s >= 1 -> ypart + (s-1) * nnz); maps_reduce builds the launch that adds
// the partial sums into y (tasks2 / segs2 / tiles2 of `out`).
void maps_chunk(const MapCtx& cx, int t0, int t1, bool first_chunk, double* Tbuf, int S, double* ypart, int64_t nnz,
                MapChunkOut& out, MapAlloc alloc, void (*dealloc)(void*), cudaStream_t st);
void maps_reduce(const MapCtx& cx, int S, double* ypart, int64_t nnz, MapChunkOut& out, MapAlloc alloc,
                 void (*dealloc)(void*), cudaStream_t st);

}  // namespace dmrg
