// nbreg_api.cu -- the C ABI of include/nbreg.h: context, argument checks, launch planning, launches.
// Every step of the path runs in the kernels of predict.cuh / force.cuh / gather.cuh; nothing here computes.
#include "../../include/nbreg.h"

#include <cstdio>
#include <cstring>
#include <new>

#include "force.cuh"
#include "gather.cuh"
#include "nbreg_common.cuh"
#include "predict.cuh"

using namespace nbreg;

namespace {

thread_local char g_errbuf[256] = "";

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return NB_E_CUDA;
}
#define NB_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

// Launch plan of the force kernel: CTA shape and j-split.
struct Plan {
    int rows_per_cta;  // IB = 32 * warps * ipt
    int ipt;
    int warps;
    int jt;            // j per shared-memory tile
    int n_chunks;      // S
    int tiles_per_chunk;
    int n_tiles;
    int grid_x;
};

struct WorkspaceLayout {
    size_t packed_off, packed_bytes;
    size_t psum_off, psum_bytes;
    size_t pcnt_off, pcnt_bytes;
    size_t plist_off, plist_bytes;
    size_t total;
};

WorkspaceLayout layout(int64_t n_max, int64_t n_i_max, int32_t cap) {
    WorkspaceLayout w{};
    const int64_t n_pad = round_up(n_max, kJPad);
    // rows x chunks of the j-split path never exceed kRowChunkLimit (make_plan), nor is the path taken for
    // blocks so large that one chunk per row suffices
    const int64_t rc = kRowChunkLimit;
    (void)n_i_max;
    size_t off = 0;
    auto place = [&](size_t bytes, size_t& o, size_t& b) {
        o = off;
        b = bytes;
        off += (size_t)round_up((int64_t)bytes, 256);
    };
    place((size_t)n_pad * kBytesPerJ, w.packed_off, w.packed_bytes);
    place((size_t)rc * 6 * sizeof(double), w.psum_off, w.psum_bytes);
    place((size_t)rc * sizeof(int32_t), w.pcnt_off, w.pcnt_bytes);
    place((size_t)rc * (size_t)cap * sizeof(int32_t), w.plist_off, w.plist_bytes);
    w.total = off;
    return w;
}

}  // namespace

struct nb_ctx {
    int device = 0;
    int num_sms = 0;
    int64_t n_max = 0, n_i_max = 0;
    int32_t cap = 0;
    unsigned char* ws = nullptr;
    bool ws_owned = false;
    WorkspaceLayout lay{};
    // registered j-state (device pointers owned by the caller)
    int64_t n = 0;
    const double *x0 = nullptr, *v0 = nullptr, *a0 = nullptr, *j0 = nullptr, *m = nullptr, *t0 = nullptr;
    bool predicted = false;
    double t_pred = 0.0;
    // options
    int64_t opt_j_split = 0, opt_i_block = 0, opt_warp_target = 0;
    // last launch
    int64_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // host path: device mirrors owned by the context
    cudaStream_t hstream = nullptr;
    unsigned char* hbuf = nullptr;
    size_t hbuf_bytes = 0;
};

namespace {

Plan make_plan(const nb_ctx* c, int32_t n_i) {
    Plan p{};
    const int64_t n_pad = round_up(c->n, kJPad);
    const int64_t sms = c->num_sms > 0 ? c->num_sms : 148;
    const int64_t min_ctas = 6 * sms;  // enough CTAs for the hardware scheduler to balance the SMs
    int ib;
    if (c->opt_i_block) {
        ib = (int)c->opt_i_block;
    } else if (n_i >= 256 * min_ctas) {
        ib = 256;
    } else if (n_i >= 128 * min_ctas) {
        ib = 128;
    } else if (n_i >= 64 * min_ctas) {
        ib = 64;
    } else {
        ib = 32;
    }
    switch (ib) {
        case 32: p.ipt = 1; p.warps = 1; p.jt = 64; break;
        case 64: p.ipt = 1; p.warps = 2; p.jt = 128; break;
        case 128: p.ipt = 1; p.warps = 4; p.jt = 128; break;
        case 256: p.ipt = 1; p.warps = 8; p.jt = 256; break;
        default: p.ipt = 2; p.warps = 8; p.jt = 256; ib = 512; break;
    }
    p.rows_per_cta = ib;
    p.grid_x = (int)((n_i + ib - 1) / ib);
    p.n_tiles = (int)(n_pad / p.jt);
    // j-split: when the block has too few warps to fill the machine, split the j-range
    const int64_t warps_total = (n_i + 31) / 32;
    const int64_t warp_target = c->opt_warp_target ? c->opt_warp_target : 16 * sms;
    int64_t S = 1;
    if (c->opt_j_split) {
        S = c->opt_j_split;
    } else if (warps_total < warp_target) {
        S = (warp_target + warps_total - 1) / warps_total;
    }
    const int64_t rows_pad = (int64_t)p.grid_x * ib;
    if (S > 1 && rows_pad * S > kRowChunkLimit) S = kRowChunkLimit / rows_pad;
    if (S > p.n_tiles) S = p.n_tiles;
    if (S < 1) S = 1;
    p.tiles_per_chunk = (int)((p.n_tiles + S - 1) / S);
    p.n_chunks = (p.n_tiles + p.tiles_per_chunk - 1) / p.tiles_per_chunk;
    return p;
}

template <int IPT, int WARPS, int JT, int MINB>
int launch_force(nb_ctx* c, const Plan& p, const ForceArgs& fa, cudaStream_t st) {
    auto kern = force_kernel<IPT, WARPS, JT, MINB>;
    const size_t smem = 2 * (size_t)JT * kBytesPerJ + 2 * sizeof(uint64_t);
    NB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, smem);
    c->info[7] = per_sm;
    dim3 grid(p.grid_x, p.n_chunks);
    kern<<<grid, WARPS * 32, smem, st>>>(fa);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

int run_predict(nb_ctx* c, double t, cudaStream_t st, double* xp_out, double* vp_out) {
    PredictArgs pa{};
    pa.n = c->n;
    pa.n_pairs = round_up(c->n, kJPad) / 2;
    pa.x0 = c->x0; pa.v0 = c->v0; pa.a0 = c->a0; pa.j0 = c->j0; pa.m = c->m; pa.t0 = c->t0;
    pa.t = t;
    pa.packed = reinterpret_cast<float4*>(c->ws + c->lay.packed_off);
    pa.xp_out = xp_out;
    pa.vp_out = vp_out;
    const int threads = 256;
    if (xp_out) {
        const int64_t pairs = (c->n + 1) / 2;
        pa.n_pairs = pairs;
        predict_kernel<true><<<(unsigned)((pairs + threads - 1) / threads), threads, 0, st>>>(pa);
    } else {
        predict_kernel<false><<<(unsigned)((pa.n_pairs + threads - 1) / threads), threads, 0, st>>>(pa);
    }
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" {

int nb_version(void) { return 100; }

const char* nb_strerror(int code) {
    switch (code) {
        case NB_OK: return "ok";
        case NB_E_INVAL: return "invalid argument";
        case NB_E_STATE: return "call out of order (no j-state registered / nothing predicted yet)";
        case NB_E_NOMEM: return "workspace too small or device allocation failed";
        case NB_E_CUDA: return g_errbuf[0] ? g_errbuf : "CUDA error";
        default: return "unknown error code";
    }
}

size_t nb_workspace_bytes(int64_t n_max, int64_t n_i_max, int32_t nbr_cap) {
    if (n_max < 1 || n_i_max < 0 || nbr_cap < 1 || n_max > 0x7fffff00LL || n_i_max > 0x7fffffffLL) return 0;
    return layout(n_max, n_i_max, nbr_cap).total;
}

int nb_create(nb_ctx** out, int device, int64_t n_max, int64_t n_i_max, int32_t nbr_cap, void* dev_workspace,
              size_t workspace_bytes) {
    if (!out) return NB_E_INVAL;
    *out = nullptr;
    const size_t need = nb_workspace_bytes(n_max, n_i_max, nbr_cap);
    if (need == 0) return NB_E_INVAL;
    if (dev_workspace && workspace_bytes < need) return NB_E_NOMEM;
    if (dev_workspace && (reinterpret_cast<uintptr_t>(dev_workspace) & 255u)) return NB_E_INVAL;
    int ndev = 0;
    NB_CUDA(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(device));
    nb_ctx* c = new (std::nothrow) nb_ctx();
    if (!c) return NB_E_NOMEM;
    c->device = device;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    c->n_max = n_max;
    c->n_i_max = n_i_max;
    c->cap = nbr_cap;
    c->lay = layout(n_max, n_i_max, nbr_cap);
    if (dev_workspace) {
        c->ws = static_cast<unsigned char*>(dev_workspace);
    } else {
        if (cudaMalloc(&c->ws, need) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return NB_E_NOMEM;
        }
        c->ws_owned = true;
    }
    *out = c;
    return NB_OK;
}

int nb_destroy(nb_ctx* c) {
    if (!c) return NB_OK;
    cudaSetDevice(c->device);
    if (c->hstream) {
        cudaStreamSynchronize(c->hstream);
        cudaStreamDestroy(c->hstream);
    }
    if (c->hbuf) cudaFree(c->hbuf);
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    delete c;
    return NB_OK;
}

int nb_set_j(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0, const double* j0,
             const double* m, const double* t0) {
    if (!c || !x0 || !v0 || !a0 || !j0 || !m || !t0) return NB_E_INVAL;
    if (n < 1 || n > c->n_max) return NB_E_INVAL;
    if (!aligned16(x0) || !aligned16(v0) || !aligned16(a0) || !aligned16(j0) || !aligned16(m) || !aligned16(t0))
        return NB_E_INVAL;  // the predictor reads 16-byte vectors
    c->n = n;
    c->x0 = x0; c->v0 = v0; c->a0 = a0; c->j0 = j0; c->m = m; c->t0 = t0;
    c->predicted = false;
    return NB_OK;
}

int nb_predict_j(nb_ctx* c, double t, void* stream) {
    if (!c) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    int rc = run_predict(c, t, static_cast<cudaStream_t>(stream), nullptr, nullptr);
    if (rc != NB_OK) return rc;
    c->predicted = true;
    c->t_pred = t;
    return NB_OK;
}

int nb_get_predicted(nb_ctx* c, double* xp, double* vp, void* stream) {
    if (!c || !xp || !vp) return NB_E_INVAL;
    if (c->n < 1 || !c->predicted) return NB_E_STATE;
    if (!aligned16(xp) || !aligned16(vp)) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    return run_predict(c, c->t_pred, static_cast<cudaStream_t>(stream), xp, vp);
}

int nb_regular_force(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const double* r_s, double t, double* acc,
                     double* jerk, int32_t* nbr_count, int32_t* nbr_list, int32_t* n_overflow, void* stream) {
    if (!c || !n_overflow) return NB_E_INVAL;
    if (n_i < 0 || n_i > c->n_i_max) return NB_E_INVAL;
    if (n_i > 0 && (!i_idx || !r_s || !acc || !jerk || !nbr_count || !nbr_list)) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int launches = 0;
    if (!c->predicted || c->t_pred != t) {  // the fused call: S1 first, same stream
        int rc = nb_predict_j(c, t, stream);
        if (rc != NB_OK) return rc;
        ++launches;
    }
    NB_CUDA(cudaMemsetAsync(n_overflow, 0, sizeof(int32_t), st));
    if (n_i == 0) {
        c->info[5] = launches;
        return NB_OK;
    }
    const Plan p = make_plan(c, n_i);
    ForceArgs fa{};
    fa.packed = reinterpret_cast<const float4*>(c->ws + c->lay.packed_off);
    fa.n = (int32_t)c->n;
    fa.n_tiles = p.n_tiles;
    fa.tiles_per_chunk = p.tiles_per_chunk;
    fa.n_chunks = p.n_chunks;
    fa.n_i = n_i;
    fa.cap = c->cap;
    fa.i_idx = i_idx;
    fa.r_s = r_s;
    fa.acc = acc; fa.jerk = jerk; fa.nbr_count = nbr_count; fa.nbr_list = nbr_list; fa.n_overflow = n_overflow;
    fa.part_sum = reinterpret_cast<double*>(c->ws + c->lay.psum_off);
    fa.part_cnt = reinterpret_cast<int32_t*>(c->ws + c->lay.pcnt_off);
    fa.part_list = reinterpret_cast<int32_t*>(c->ws + c->lay.plist_off);
    int rc;
    switch (p.rows_per_cta) {
        case 32: rc = launch_force<1, 1, 64, 16>(c, p, fa, st); break;
        case 64: rc = launch_force<1, 2, 128, 8>(c, p, fa, st); break;
        case 128: rc = launch_force<1, 4, 128, 4>(c, p, fa, st); break;
        case 256: rc = launch_force<1, 8, 256, 2>(c, p, fa, st); break;
        default: rc = launch_force<2, 8, 256, 1>(c, p, fa, st); break;
    }
    if (rc != NB_OK) return rc;
    ++launches;
    if (p.n_chunks > 1) {
        GatherArgs ga{};
        ga.n_i = n_i; ga.n_chunks = p.n_chunks; ga.cap = c->cap;
        ga.part_sum = fa.part_sum; ga.part_cnt = fa.part_cnt; ga.part_list = fa.part_list;
        ga.acc = acc; ga.jerk = jerk; ga.nbr_count = nbr_count; ga.nbr_list = nbr_list; ga.n_overflow = n_overflow;
        const unsigned blocks = (unsigned)((n_i + kGatherWarps - 1) / kGatherWarps);
        reduce_gather_kernel<<<blocks, kGatherWarps * 32, 0, st>>>(ga);
        NB_CUDA(cudaGetLastError());
        ++launches;
    }
    c->info[0] = p.rows_per_cta; c->info[1] = p.ipt; c->info[2] = p.n_chunks; c->info[3] = p.grid_x;
    c->info[4] = p.n_chunks; c->info[5] = launches; c->info[6] = p.jt;
    return NB_OK;
}

int nb_regular_force_host(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0,
                          const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                          const double* r_s, double t, double* acc, double* jerk, int32_t* nbr_count,
                          int32_t* nbr_list, int32_t* n_overflow) {
    if (!c || !x0 || !v0 || !a0 || !j0 || !m || !t0 || !n_overflow) return NB_E_INVAL;
    if (n < 1 || n > c->n_max || n_i < 0 || n_i > c->n_i_max) return NB_E_INVAL;
    if (n_i > 0 && (!i_idx || !r_s || !acc || !jerk || !nbr_count || !nbr_list)) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    if (!c->hstream) NB_CUDA(cudaStreamCreateWithFlags(&c->hstream, cudaStreamNonBlocking));
    // device mirrors, carved from one allocation sized for n_max / n_i_max / cap
    const size_t nmax = (size_t)c->n_max, imax = (size_t)c->n_i_max;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off += (size_t)round_up((int64_t)bytes, 256); return o; };
    const size_t o_x0 = carve(nmax * 24), o_v0 = carve(nmax * 24), o_a0 = carve(nmax * 24), o_j0 = carve(nmax * 24);
    const size_t o_m = carve(nmax * 8), o_t0 = carve(nmax * 8);
    const size_t o_idx = carve(imax * 4), o_rs = carve(imax * 8);
    const size_t o_acc = carve(imax * 24), o_jrk = carve(imax * 24), o_cnt = carve(imax * 4);
    const size_t o_lst = carve(imax * (size_t)c->cap * 4), o_ovf = carve(256);
    if (!c->hbuf) {
        if (cudaMalloc(&c->hbuf, off) != cudaSuccess) {
            cudaGetLastError();
            return NB_E_NOMEM;
        }
        c->hbuf_bytes = off;
    }
    unsigned char* b = c->hbuf;
    cudaStream_t st = c->hstream;
    const size_t nn = (size_t)n, ni = (size_t)n_i;
    NB_CUDA(cudaMemcpyAsync(b + o_x0, x0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_v0, v0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_a0, a0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_j0, j0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_m, m, nn * 8, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_t0, t0, nn * 8, cudaMemcpyHostToDevice, st));
    if (n_i > 0) {
        NB_CUDA(cudaMemcpyAsync(b + o_idx, i_idx, ni * 4, cudaMemcpyHostToDevice, st));
        NB_CUDA(cudaMemcpyAsync(b + o_rs, r_s, ni * 8, cudaMemcpyHostToDevice, st));
    }
    int rc = nb_set_j(c, n, (const double*)(b + o_x0), (const double*)(b + o_v0), (const double*)(b + o_a0),
                      (const double*)(b + o_j0), (const double*)(b + o_m), (const double*)(b + o_t0));
    if (rc != NB_OK) return rc;
    rc = nb_regular_force(c, n_i, (const int32_t*)(b + o_idx), (const double*)(b + o_rs), t, (double*)(b + o_acc),
                          (double*)(b + o_jrk), (int32_t*)(b + o_cnt), (int32_t*)(b + o_lst), (int32_t*)(b + o_ovf),
                          st);
    if (rc != NB_OK) return rc;
    if (n_i > 0) {
        NB_CUDA(cudaMemcpyAsync(acc, b + o_acc, ni * 24, cudaMemcpyDeviceToHost, st));
        NB_CUDA(cudaMemcpyAsync(jerk, b + o_jrk, ni * 24, cudaMemcpyDeviceToHost, st));
        NB_CUDA(cudaMemcpyAsync(nbr_count, b + o_cnt, ni * 4, cudaMemcpyDeviceToHost, st));
        NB_CUDA(cudaMemcpyAsync(nbr_list, b + o_lst, ni * (size_t)c->cap * 4, cudaMemcpyDeviceToHost, st));
    }
    NB_CUDA(cudaMemcpyAsync(n_overflow, b + o_ovf, 4, cudaMemcpyDeviceToHost, st));
    NB_CUDA(cudaStreamSynchronize(st));
    // the registered pointers are the context's own mirrors; they stay valid, but a new host call overwrites them
    return NB_OK;
}

int nb_set_option(nb_ctx* c, const char* key, int64_t value) {
    if (!c || !key || value < 0) return NB_E_INVAL;
    if (!strcmp(key, "j_split")) {
        c->opt_j_split = value;
        return NB_OK;
    }
    if (!strcmp(key, "i_block")) {
        if (value != 0 && value != 32 && value != 64 && value != 128 && value != 256 && value != 512)
            return NB_E_INVAL;
        c->opt_i_block = value;
        return NB_OK;
    }
    if (!strcmp(key, "warp_target")) {
        c->opt_warp_target = value;
        return NB_OK;
    }
    return NB_E_INVAL;
}

int nb_last_launch_info(const nb_ctx* c, int64_t info[8]) {
    if (!c || !info) return NB_E_INVAL;
    for (int k = 0; k < 8; ++k) info[k] = c->info[k];
    return NB_OK;
}

}  // extern "C"
