// Host orchestrator of the B200 DMRG hot path: block-sparse operator storage on the device, plans (block maps)
// for the grouped FP64 GEMM kernel, environments, H_eff, Davidson, truncation, sweep and RDM drivers.
// All arithmetic on tensors runs in the CUDA kernels declared in kernels.hpp; this layer only builds integer
// block maps and launch descriptors (DESIGN.md "Kernels" and "Data layout").
#pragma once
#include <cuda_runtime_api.h>

#include <map>
#include <memory>
#include <stdexcept>
#include <string>
#include <unordered_map>
#include <vector>

#include "kernels.hpp"
#include "sym.hpp"

namespace dmrg {

struct Error : std::runtime_error {
    int code;
    Error(int code_, const std::string& msg) : std::runtime_error(msg), code(code_) {}
};
void cuda_check(cudaError_t e, const char* what);

// ---- device memory ------------------------------------------------------------------------------------------------
extern int64_t g_device_bytes;
void* dev_alloc(size_t bytes);
void dev_free(void* p);

template <class T>
struct DevVec {
    T* p = nullptr;
    size_t n = 0;
    DevVec() {}
    DevVec(const DevVec&) = delete;
    DevVec& operator=(const DevVec&) = delete;
    DevVec(DevVec&& o) noexcept : p(o.p), n(o.n) { o.p = nullptr; o.n = 0; }
    DevVec& operator=(DevVec&& o) noexcept { release(); p = o.p; n = o.n; o.p = nullptr; o.n = 0; return *this; }
    ~DevVec() { release(); }
    void release() { if (p) dev_free(p); p = nullptr; n = 0; }
    void alloc(size_t n_) { release(); n = n_; if (n) p = (T*)dev_alloc(n * sizeof(T)); }
    void upload_raw(const T* src, size_t count, cudaStream_t st) {
        if (count > n) alloc(count);
        if (count) cuda_check(cudaMemcpyAsync(p, src, count * sizeof(T), cudaMemcpyHostToDevice, st), "upload");
    }
    void upload(const std::vector<T>& v, cudaStream_t st) {
        if (v.size() > n) alloc(v.size());
        if (!v.empty()) cuda_check(cudaMemcpyAsync(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st), "upload");
    }
};

// ---- block-sparse bases and tensors -------------------------------------------------------------------------------
struct Sector { int n, s, d; };
typedef std::vector<Sector> Basis;               // sorted ascending by (n, s)
int find_sector(const Basis& b, int n, int s);    // index or -1
inline int pad2(int d) { return (d + 1) & ~1; }

struct SiteTensor {                               // one MPS site, device-resident
    struct Blk { int l, s, r, rows, cols, ld; double* ptr; };   // dense [rows x cols], row stride ld (even)
    std::vector<Blk> blocks;                      // ordered by (l, s)
    std::vector<int> lookup;                      // [l*4+s] -> block index or -1
    DevVec<double> data;
    int64_t nnz = 0;                              // doubles of storage including padding
    char gauge = 'R';
    const Blk* get(int l, int s) const { int j = lookup[l * 4 + s]; return j < 0 ? nullptr : &blocks[j]; }
};
struct MPS {
    int k = 0, n_elec = 0, two_sz = 0;
    std::vector<Basis> bonds;                     // k+1
    std::vector<SiteTensor> sites;                // k
};
// allocate a site tensor with all blocks (l, s) -> r allowed by the two bases
void make_site_tensor(SiteTensor& t, const Basis& bl, const Basis& br);

// ---- launch descriptors --------------------------------------------------------------------------------------------
struct GemmBatch {                                // host-side builder of one grouped-GEMM launch
    std::vector<Task> tasks;
    std::vector<Seg> segs;
    std::vector<int> seg_task;                    // owning task of each seg (segs may arrive in any order)
    double flops = 0.0;
    int add_task(double* C, int ldc, int M, int N, int flags);
    void add_seg(int task, const double* A, int lda, const double* B, int ldb, int K, int flags, double alpha);
    bool empty() const { return tasks.empty(); }
};
struct GemmLaunch {                               // device-resident descriptors, reusable
    DevVec<Task> tasks;
    DevVec<Seg> segs;
    DevVec<Tile> tiles;
    DevVec<int> counter;                          // dynamic tile counter of the persistent kernel
    int ntiles = 0;
    bool aligned = false;                         // every GEMM operand 16-byte aligned, even ld: bulk-copy kernel
    double flops = 0.0;
};
// Growable pinned host buffer: descriptor tables are written straight into it and uploaded by DMA (a pageable source is
// staged by the driver at a fraction of the rate, and fresh 100 MB vectors page-fault on every call).
struct PinnedBuf {
    void* p = nullptr;
    size_t bytes = 0;
    void* get(size_t n);
    PinnedBuf() {}
    PinnedBuf(const PinnedBuf&) = delete;
    PinnedBuf& operator=(const PinnedBuf&) = delete;
    ~PinnedBuf();
};
struct FinalizeScratch {                          // reused by every finalize() of a context (capacity is kept)
    PinnedBuf segs, tiles, tasks;
    std::vector<int> off, idx, fill, ntile, bucket;
    std::vector<double> weight, tw;
    std::vector<Tile> raw;
    std::vector<size_t> hist;
};
struct Engine;
void finalize(GemmBatch& b, GemmLaunch& out, Engine& eng);   // sort segs by task, build tiles, upload
void run(const GemmLaunch& l, Engine& eng, cudaStream_t st = nullptr);   // st: stream override (default eng.stream)
void run_once(GemmBatch& b, Engine& eng);                    // finalize + run + release (synchronises)
double run_once_ms(GemmBatch& b, Engine& eng);               // same, returns the kernel's device time (CUDA events)

// ---- operator storage ----------------------------------------------------------------------------------------------
struct OpClass {                                  // block structure shared by all operators with one label shift
    int dn, ds;
    std::vector<int> out;                         // per in-sector: out-sector index or -1
    std::vector<int> inv;                         // per out-sector: in-sector index or -1
    std::vector<int64_t> off;                     // per in-sector: offset of the dense [d_out x d_in] block
    int64_t nnz = 0, ld = 0;                      // ld = nnz rounded up to even (16-byte aligned rows of a stack)
};
struct Stack {                                    // operators of one (kind, class), rows of a [n x ld] matrix
    int kind, cls;
    double* base = nullptr;
    std::vector<Label> members;
    int alloc = -1;                               // index into Block::allocs (-1: temporary storage)
    int64_t alloc_off = 0;                        // offset of the stack inside that allocation (doubles)
};
// Pinned host memory for spilled environment blocks (SURVEY.md 7 hard part 5): regions are reused across passes and
// sweeps because pinning is slow (seconds per 10 GB); freed with the context.
struct HostPool {
    struct Region { double* p; size_t doubles; bool used; };
    std::vector<Region> regions;
    int64_t bytes = 0;
    double* get(size_t doubles);
    void put(double* p);
    void clear();
    ~HostPool() { clear(); }
};
struct BlockAlloc { double* dev = nullptr; size_t doubles = 0; double* host = nullptr; };
struct OpRef { int cls = -1; double* ptr = nullptr; int stack = -1, row = -1; };

struct Block {
    char side;                                    // 'L': sites [0,b)   'R': sites [b,k)
    int b, k;
    char mode;                                    // 'N': normal two-index operators A, B   'C': complementary Pt, Q
    Basis basis;
    std::vector<OpClass> classes;
    std::vector<Stack> stacks;
    std::unordered_map<uint32_t, OpRef> ops;
    std::vector<BlockAlloc> allocs;               // persistent storage: on the device, or spilled to pinned host memory
    std::vector<void*> temp_allocs;               // temporaries of make_temps
    bool spilled = false;                         // storage lives in allocs[].host; restore() before use
    cudaEvent_t spill_done = nullptr;             // device copies may be freed once this event has completed
    HostPool* pool = nullptr;
    std::vector<uint32_t> temp_keys;
    Block(char side, int b, int k, const Basis& basis, char mode);
    ~Block();
    int g() const { return side == 'L' ? 1 : -1; }
    std::vector<int> inside() const;
    std::vector<int> outside() const;
    bool has(const Label& l) const { return ops.find(l.key()) != ops.end(); }
    const OpRef& get(const Label& l) const;
    int class_of(int dn, int ds);                 // find or create
    int label_class(const Label& l);              // class of the stored (untransposed) operator
    // allocate storage for a set of new operators grouped into (kind, class) stacks; temp: freed by drop_temps()
    void allocate(const std::vector<Label>& labels, bool temp);
    void drop_temps();
    void drop_kind(int kind);                     // forget operators of a kind (storage is released with the block)
    int64_t bytes() const;
    int64_t bytes_ = 0;
    // environment-stack memory path: asynchronous device -> pinned host copy on `copy_stream`; finish_spill() waits for
    // it and frees the device storage; restore() brings the block back and re-derives every operator pointer
    void spill(HostPool& pool, cudaStream_t copy_stream);
    void finish_spill();
    void restore(cudaStream_t st);
};

// a dense block of an operator as the GEMM kernel sees it
struct OpBlockView { int out; const double* ptr; int ld; bool trans; int rows, cols; };
// block of (op, trans) acting on in-sector `in`: returns false if absent.  View: matrix [d_out x d_in] =
// stored (ld = d_in) or stored^T (stored [d_in x d_out], ld = d_out, trans = true)
bool op_block(const Block& blk, const OpRef& op, bool trans, int in, OpBlockView& v);

struct LinItem { double coef; Label src; int stack = -1, row = -1; };   // stack / row: optional hint (skips the label lookup)
struct LinSpec { Label dst; std::vector<LinItem> items; };
// dst = (accumulate ? dst : 0) + sum coef * src for every spec, as one stack GEMM per (kind, class) pair
void lincomb(Block& blk, const std::vector<LinSpec>& specs, bool accumulate, Engine& eng);

// temporaries on X needed to enlarge it by `dot` (far = outside orbitals whose S_P is needed)
void make_temps(const Ham& ham, Block& X, const Dot& dot, const std::vector<int>& far, Engine& eng);
std::unique_ptr<Block> empty_block(char side, int k, const MPS& mps);
// one blocking step with the tensor of the neighbouring site (fused form-and-rotate)
std::unique_ptr<Block> grow(Block& X, const Ham& ham, const MPS& mps, char new_mode, Engine& eng);
// blocking step that keeps only a+_P of every inside orbital and A_PQ, B_PS of the pairs whose two SITES both lie in
// [pair_lo, pair_hi) (empty range: one-index operators only): what the RDM pass needs
std::unique_ptr<Block> grow_normal(Block& X, const Ham& ham, const Basis& new_basis, const SiteTensor& tensor,
                                   int pair_lo, int pair_hi, Engine& eng);
BlockInfo block_info(const Block& b);

// ---- H_eff ---------------------------------------------------------------------------------------------------------
struct PsiBlock { int l, ab, r, rows, cols; int64_t off; int64_t poff; };   // poff: offset in the padded (even ld) copy
typedef DiagItemK DiagItem;                      // null pointer = identity factor
struct HeffPlan {
    int bond = -1;
    std::vector<PsiBlock> layout;
    std::vector<int> lookup;                      // [l*16+ab] -> layout index or -1
    int64_t nnz = 0;
    struct Chunk { GemmLaunch p1, p2; };
    std::vector<Chunk> chunks;
    int split = 1;                                // split-K parts of phase 2 (device-built maps): parts >= 1 go to ypart
    DevVec<double> ypart;                         // (split - 1) x nnz partial sums
    GemmLaunch reduce;                            // y += sum of the partial sums, in part order
    DevVec<double> T, T2, xbuf, ybuf, xpad;       // T / T2: intermediates of even / odd chunks (double buffered)           // xpad: x with even leading dimensions, 16-byte aligned blocks
    int64_t nnz_pad = 0;
    DevVec<int64_t> blk_poff;
    DevVec<DiagItem> diag_items;
    DevVec<int> diag_ptr;                         // per psi block range into diag_items
    DevVec<int64_t> blk_off;
    DevVec<int> blk_rows, blk_cols;
    double f_alg = 0, f_exec = 0, b_alg = 0;
    int64_t nterms = 0, ngemm = 0;
    Block* X = nullptr;                           // block carrying temporaries
    std::vector<cudaEvent_t> ev_p1, ev_p2;        // per chunk: phase 1 done / phase 2 done
    cudaEvent_t ev_in = nullptr;                  // x is ready on the main stream
    ~HeffPlan();                                  // drops the temporaries on X
};
void psi_layout(const Basis& bl, const Basis& br, std::vector<PsiBlock>& layout, std::vector<int>& lookup,
                int64_t& nnz);
std::unique_ptr<HeffPlan> build_heff(const Ham& ham, Block& LB, Block& RB, int i, Engine& eng);
void heff_apply(HeffPlan& p, const double* x_dev, double* y_dev, Engine& eng);
void heff_diag(HeffPlan& p, double* d_dev, Engine& eng);

// ---- engine --------------------------------------------------------------------------------------------------------
struct Options {
    double davidson_tol = 1e-7;
    int davidson_max_iter = 100, davidson_max_subspace = 20;
    double sv_floor = 1e-10, cluster_rel_gap = 1e-6;
    int device_id = 0;
    int64_t workspace_bytes = 0;
    int64_t hbm_budget_bytes = 0;                 // device bytes the environment stack of a sweep may hold (0 = automatic)
    int64_t host_budget_bytes = 0;                // pinned host bytes for spilled checkpoints (0 = automatic: 64 GiB)
    int host_spill = 0;                           // 1: environment checkpoints may live in pinned host memory
    int env_stride = 0;                           // checkpoint spacing of the environment stack (0 = automatic, 1 = keep all)
    int env_stride2 = 0;                          // second checkpoint level inside a segment (used with an explicit env_stride)
    double dbss_eps = 0.0;                        // > 0: dynamic block state selection, truncation error target per bond
    int dbss_dmin = 0;                            // DBSS lower bound on the kept states
    int split_k = 0;                              // split-K parts of phase 2 of H_eff psi (0 = automatic)
    int svd_qr = 0;                               // 1: QR-iteration SVD (gesvd) instead of one-sided Jacobi (gesvdj)
    int eigensolver = 0;                          // 0: Davidson, 1: Lanczos
    int rdm_split = -1;                           // site kh separating the two centre rules of the RDM pass (-1: k/2)
};
struct BondRecord {
    int bond, forward;
    double energy, residual, trunc_err;
    int n_matvec, kept, nsectors, converged;
    int64_t nnz;
    double f_alg, seconds, seconds_matvec;
};
struct Engine {
    Ham ham;
    Options opt;
    int k = 0, n_elec = 0, two_sz = 0, bsw = 0;
    cudaStream_t stream = nullptr;                // the library's own stream
    cudaStream_t stream2 = nullptr;               // second stream: phase 2 of H_eff psi runs beside the next chunk's phase 1
    MPS mps;
    bool have_mps = false;
    std::map<int, std::unique_ptr<Block>> L, R;   // by bond
    std::unique_ptr<HeffPlan> plan;
    int64_t launches = 0;
    double flops_total = 0;                       // unpadded flops of every grouped-GEMM launch since creation
    std::string last_error;
    SvdWork* svd = nullptr;
    DevVec<double> red_scratch;                   // partial sums of the two-stage reductions (per context)
    std::vector<SvdWork*> svd_pool;               // extra cuSOLVER handles on their own streams: sector SVDs run concurrently
    std::vector<cudaStream_t> svd_streams;
    void ensure_svd_pool(int n);
    FinalizeScratch fin;
    int host_threads = 1;                         // size of the one OpenMP team every host-parallel region uses (a changing
                                                  // team size makes libgomp rebuild its thread pool at every region)
    double rdm_seconds = 0, rdm_bytes = 0, rdm_flops = 0, rdm_host_seconds = 0, rdm_grow_seconds = 0, rdm_gemm_ms = 0;
    double rdm_stream_bytes = 0;                  // bytes of the launches of the HBM-bound streaming kernel alone
    double t_plan = 0, t_davidson = 0, t_split = 0, t_grow = 0, t_matvec = 0;   // phase seconds of the last sweep
    double rdm_stream_ms = 0;                     // device time of the operator-streaming kernels (E = Stack M^T) alone
    bool keep_env_stack = true;
    // environment-stack memory path of dmrg_sweep (row "m"): checkpoints every env_stride bonds, the blocks between two
    // checkpoints are recomputed when a pass enters that segment; checkpoints optionally spilled to pinned host memory
    int env_stride = 1, env_stride2 = 1;
    bool env_spill = false;
    int64_t ws_cap = 0;                           // doubles: cap of a T buffer chosen by the policy when the stack is checkpointed (0: none)
    HostPool host_pool;
    cudaStream_t copy_stream = nullptr;
    std::vector<Block*> pending_spills;
    double t_spill_wait = 0, t_restore = 0, t_regrow = 0, spill_bytes = 0, restore_bytes = 0, t_env = 0;
    int env_D = 0;
    int64_t env_peak_bytes = 0, env_est_total = 0, env_est_max = 0;
    void plan_env_policy(int D);                  // choose env_stride / env_spill from the options and the memory estimate
    void finish_spills();
    Block& need_left(int b);                      // device-resident L_b (restored or regrown from the nearest checkpoint)
    Block& need_right(int b);
    void retire_left(int b);                      // L_b has produced L_{b+1}: keep as checkpoint (spill) or erase
    void retire_right(int b);
    void build_right_stack();                     // R_k .. R_2 under the policy (start of the first sweep)
    bool sweep_ready = false;                     // environments consistent with the sweep position
    bool host_maps = false;                       // dmrg_options.host_maps: build the H_eff block maps on the host (A/B testing)
    bool trace = false;                           // DMRG_B200_TRACE=1: print every grouped-GEMM launch's device time
    bool force_generic_gemm = false;              // dmrg_options.generic_gemm: always the cp.async kernel (A/B testing)
    char mode_L(int b) const { return b <= bsw ? 'N' : 'C'; }
    char mode_R(int b) const { return b >= bsw + 3 ? 'N' : 'C'; }
    int64_t t_capacity() const;                   // doubles available for intermediates
    void invalidate() { plan.reset(); pending_spills.clear(); L.clear(); R.clear(); sweep_ready = false; }   // the plan owns temporaries on a block
    void ensure_left(int i);                      // L_0 .. L_i present
    void ensure_right(int j);                     // R_k .. R_j present
    void prepare_bond(int i);
};

// Davidson, decomposition, sweep (sweep.cpp)
struct DavidsonResult { double theta, residual; int n_matvec; bool converged; double seconds_matvec; };
DavidsonResult davidson(HeffPlan& p, double* x_dev /*in: guess, out: eigenvector*/, Engine& eng);
DavidsonResult lanczos(HeffPlan& p, double* x_dev /*in: guess, out: eigenvector*/, Engine& eng);
void two_site_tensor(const MPS& mps, int i, const HeffPlan& p, double* theta_dev, Engine& eng);
// SVD + truncation of the two-site vector; replaces sites i, i+1 and bond i+1 of the MPS (reading S14)
void split_theta(MPS& mps, int i, const HeffPlan& p, const double* theta_dev, int D, bool forward, Engine& eng,
                 double& trunc_err, int& kept, int& nsectors);
int sweep(Engine& eng, int D, std::vector<BondRecord>& recs, double& seconds);
// RDM pass (rdm.cpp)
void rdm12(Engine& eng, double* gamma_host, double* Gamma_host);

}  // namespace dmrg
