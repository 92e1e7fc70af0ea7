// fx_internal.h -- host-side state shared by the translation units of libfx.so (not part of the ABI).
#ifndef FX_INTERNAL_H
#define FX_INTERNAL_H

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/fx.h"
#include "fx_dg.cuh"
#include "fx_dgt.cuh"
#include "fx_exdot.cuh"
#include "fx_tables.h"

#define FX_NUM_SMS_DEFAULT 148

struct FxFuncInfo { const void* f; int block; size_t smem; int occ; };

// The opaque fx_ctx of include/fx.h.  One context = one device, one stream, its own scratch: exact-dot digits and ticket, result
// slots, CG work vectors and scalars, staging buffers, launch-shape overrides, per-kernel attribute / occupancy cache.
// Contexts share nothing mutable, so different contexts may be used from different threads and streams at the same time;
// ONE context must be used by one thread at a time (its kernels are stream-ordered and share the digit scratch).
struct fx_ctx {
    bool ready;
    int device, num_sms;
    FxFuncInfo fcache[128]; int nfcache;   // kernels whose shared-memory attribute is set on this device, with their occupancy
    cudaStream_t stream;
    ExGlobal ex;                 // device scratch of the exact dot
    double* result_dev;          // [8] scratch doubles (dot results of the synchronous calls)
    double* result_pinned;       // [8] pinned host mirror
    // launch-shape overrides (fx_set_launch): [kernel_id][0]=grid, [1]=block
    int launch[4][2];
    int cg_fused;
    int dg_path;                // 0 = automatic (CTA-tile kernels where TMA's rules allow; CG's K1: tile for P >= 4), 1 = warp-strip kernels, 2 = tile kernels, K1 too
    int cg_pdl;                 // programmatic dependent launch of the fused loop's kernels (off; environment FX_PDL=1 turns it on)
    // CG work space
    double* cg_vec; int64_t cg_cap;   // 7 vectors of cg_cap doubles
    void* cg_scal;                     // CgScal on the device
    void* cg_scal_pinned;
    double* ara_vec; int64_t ara_cap;  // six work vectors of fx_arakawa
    void* cg_pdig;                     // digit buffers of the persistent CG kernel
    void* cg_tile;                     // CgTile (fx_cg.cu): tensor maps and geometry of the tile K1 of the running solve
    cudaEvent_t cg_ev[2];
    // host staging for the *_host entry points
    double* stage[4]; int64_t stage_cap;
    cudaStream_t copy_stream;
    cudaEvent_t ev_copy[2], ev_comp[2];
    int64_t launches;
    // fx_cg_profile
    int prof_on, prof_iters, prof_cap, prof_stride;
    cudaEvent_t prof_loop[2];   // begin of iteration 0, end of the last enqueued batch
    cudaEvent_t* prof_ev;
    double prof_ms[4];
};

typedef struct fx_ctx FxCtx;
FxCtx* fx_default_ctx();                       // the calling thread's current device's default context, created on first use; NULL (and last error set) on failure
// resident CTAs per SM of kernel `f` at (block, smem) on the context's device; the first call per kernel also raises its
// dynamic shared-memory limit (and, with carveout, asks for the largest shared-memory carve-out)
int fx_func_occ(FxCtx* c, const void* f, int block, size_t smem, bool carveout = false);
// makes the context's device current for the scope of an _ex call (restores the caller's device afterwards)
struct FxDeviceGuard {
    int prev; bool switched;
    explicit FxDeviceGuard(const FxCtx* c) : prev(-1), switched(false) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~FxDeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define FX_ENTER(c, name)                                                        \
    if (!(c) || !(c)->ready) { fx_set_error("%s: null or destroyed context", name); return FX_EINVAL; } \
    FxDeviceGuard fx_guard_(c)
void fx_set_error(const char* fmt, ...);
fx_status fx_cuda_fail(cudaError_t e, const char* what);

#define FX_CUDA(call)                                           \
    do {                                                        \
        cudaError_t e_ = (call);                                \
        if (e_ != cudaSuccess) return fx_cuda_fail(e_, #call);  \
    } while (0)

static inline bool aligned16(const void* p) { return (((uintptr_t)p) & 15) == 0; }
int fx_grid_ok(const fx_grid* g);
int fx_grid_deriv_ok(const fx_grid* g);          // PER / DIR only: stand-alone derivatives and the bracket
int fx_dg_has_neumann(const DgParams* p);
int fx_dg_neu_variant(const DgParams* p, int P);
fx_status fx_make_dg_params(const fx_grid* g, int normed, DgParams* out, double* vol4_out, int Nz = 1, double lz = 0.0);   // lz > 0: 3-D product grid of Nz planes

// internal launchers (stream-ordered, no synchronisation)
fx_status fx_launch_exdot(FxCtx* c, const double* x, const double* y, int64_t n, double* result_dev);
fx_status fx_launch_exdot_part(FxCtx* c, const double* x, const double* y, int64_t m, int first, int last, double* result_dev, int mode = 0);   // mode 1: exact sum of two halves, 2: binary32 pairs
fx_status fx_launch_exsum(FxCtx* c, const double* x, int64_t n, double* result_dev);
fx_status fx_result_to_host(FxCtx* c, double* result_host);
size_t fx_dg_ring_bytes(int P, int warps, bool dirf);
void fx_dg_shape(FxCtx* c, const fx_grid* g, DgParams* p, int warps_per_sm, int* grid, int* block, int max_wpb = 4);
// CTA-tile stencil kernels (fx_dgt.cuh): eligibility (TMA's global-memory rules), tensor maps, launch geometry
bool fx_dgt_eligible(const fx_grid* g, const void* a, const void* b, const void* c2);
fx_status fx_dgt_make_map(CUtensorMap* m, const double* base, int pitch, int rows, int boxw, int boxh);
void fx_dgt_shape(FxCtx* c, const fx_grid* g, int nbx, int resident, DgtTile* t, int Nz = 1);
fx_status fx_launch_derivative(FxCtx* c, const fx_grid* g, int dir, int flux, double alpha, const double* x, double beta, double* y);
fx_status fx_launch_weights(FxCtx* c, const fx_grid* g, double* W, double* V, int Nz = 1, double lz = 0.0);
fx_status fx_launch_apply(FxCtx* c, const fx_grid* g, const double* chi, const double* x, double* y, int normed, int Nz = 1, double lz = 0.0);

#endif
