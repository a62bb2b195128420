// dkd_host.h — host-side helpers shared by the translation units of libdkd (not part of the C-ABI):
// a recorded kernel launch (so that the same launch can go to a stream, into a capture, or into the
// parameters of an instantiated graph's kernel node), the device guard, and the few context accessors the
// other .cu files need.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "dkd.h"

namespace dkd {

// One kernel launch, recorded: function, geometry and the argument VALUES (copied into `blob`; `off[i]` is
// where argument i lives).  Offsets instead of pointers keep the struct trivially copyable.
struct KLaunch {
    static constexpr int MAX_ARGS = 10;
    static constexpr int BLOB_BYTES = 768;
    const void* func;
    dim3 grid, block;
    size_t smem;
    bool pdl;                          // launch with programmatic stream serialization (the kernel calls griddepcontrol.wait)
    int nargs;
    uint16_t off[MAX_ARGS];
    alignas(64) unsigned char blob[BLOB_BYTES];   // (a CUtensorMap argument needs 64-byte alignment)

    void arg_pointers(void** argp) const {
        for (int i = 0; i < nargs; ++i) argp[i] = const_cast<unsigned char*>(blob) + off[i];
    }
};

// bytes the argument values of a kernel take in KLaunch::blob (each at its natural alignment, in order)
template <typename... T>
constexpr size_t packed_arg_bytes() {
    size_t o = 0;
    ((o = ((o + alignof(T) - 1) & ~(alignof(T) - 1)) + sizeof(T)), ...);
    return o;
}

template <typename... KArgs, typename... Args>
inline void prep(KLaunch& k, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, bool pdl, Args... args) {
    static_assert(sizeof...(KArgs) == sizeof...(Args), "argument count");
    static_assert(sizeof...(KArgs) <= KLaunch::MAX_ARGS, "too many kernel arguments");
    static_assert(packed_arg_bytes<KArgs...>() <= KLaunch::BLOB_BYTES, "kernel arguments do not fit KLaunch::blob");
    k.func = reinterpret_cast<const void*>(kern);
    k.grid = grid; k.block = block; k.smem = smem; k.pdl = pdl; k.nargs = 0;
    size_t o = 0;
    auto put = [&](auto v) {
        using T = decltype(v);
        o = (o + alignof(T) - 1) & ~(alignof(T) - 1);
        memcpy(k.blob + o, &v, sizeof(T));
        k.off[k.nargs++] = static_cast<uint16_t>(o);
        o += sizeof(T);
    };
    (put(static_cast<KArgs>(args)), ...);
}

// allow_pdl = false strips the programmatic attribute (measurement mode)
inline cudaError_t launch(const KLaunch& k, cudaStream_t st, bool allow_pdl) {
    if (!k.func) return cudaErrorInvalidValue;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = k.grid; cfg.blockDim = k.block; cfg.dynamicSmemBytes = k.smem; cfg.stream = st;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = (k.pdl && allow_pdl) ? 1 : 0;
    void* argp[KLaunch::MAX_ARGS];
    k.arg_pointers(argp);
    return cudaLaunchKernelExC(&cfg, k.func, argp);
}

// Every entry point runs on the context's device and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(int dev) : prev(-1), switched(false) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

}  // namespace dkd

// context accessors for the other translation units (defined in dkd_api.cu)
int dkd_ctx_device(const dkd_ctx* ctx);
int dkd_ctx_num_sms(const dkd_ctx* ctx);
int dkd_ctx_fail(dkd_ctx* ctx, int code, const char* msg, const char* detail);   // sets dkd_last_error, returns code
// context-owned device scratch buffer `slot` (0: match partials, 1: retrieval scan) of at least `bytes` bytes, grown
// with cudaMalloc when too small (not capture-safe then); NULL on failure (dkd_last_error set)
void* dkd_ctx_scratch(dkd_ctx* ctx, int slot, size_t bytes);
// shared-memory limits of k_match_tc / k_scan on the CURRENT device (dkd_match.cu); dkd_create calls it per context
cudaError_t dkd_match_setup_device();
// k_select on caller-provided candidate segments (one "image"): ranks the keys of `tpi` segments of `seg_cap` keys by
// (score desc, index asc) into sel_idx[top_k] (-1 padded) and out_count[1]; n_items bounds the indices
int dkd_internal_select(dkd_ctx* ctx, const uint64_t* cand, const int* seg_cnt, int tpi, int seg_cap, int top_k, int n_items,
                        int32_t* sel_idx, int32_t* out_count, cudaStream_t st);
