// qr_common.cuh -- shared host/device helpers of libqr (sm_100a).  Product code: nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stdio.h>
#include <stdarg.h>

#include "../../include/qr.h"

namespace qr {

// Conventions of DESIGN.md "Readings" (R4; R12).
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kAlphaMax = 0.99f;
constexpr float kPowerMin = -4.5f;
constexpr float kDilation = 0.3f;
constexpr float kJClamp = 1.3f;
constexpr int kTile = QR_TILE;

// Camera as passed to kernels (by value, in constant bank).
struct Cam {
    int32_t width, height;
    float fx, fy, cx, cy, znear;
    float w[12];
    int32_t tiles_x, tiles_y;
};

// Channel counts the tcgen05 contractions (blend_mma_kernel, backward_mma_kernel) take: they work on whole 128-channel tiles and
// let TMA pad (zeros on load, clipped on store).  The 32-channel groups of backward_mma_kernel's tensor map must be whole
// (D % 32 == 0) or there must be a single partial one (D < 32); rows must be 16-byte multiples.
inline bool tc_channels_supported(int32_t D) { return D >= 4 && D <= 512 && (D % 32 == 0 || (D < 32 && D % 4 == 0)); }

inline Cam make_cam(const qr_camera* c)
{
    Cam k;
    k.width = c->width; k.height = c->height;
    k.fx = c->fx; k.fy = c->fy; k.cx = c->cx; k.cy = c->cy; k.znear = c->znear;
    for (int i = 0; i < 12; ++i) k.w[i] = c->world_to_cam[i];
    k.tiles_x = (c->width + kTile - 1) / kTile;
    k.tiles_y = (c->height + kTile - 1) / kTile;
    return k;
}

// Thread-local error string (qr_last_error).
char* err_buf();
int fail(int code, const char* fmt, ...);
int check_cam(const qr_camera* cam);
int check_feat(int32_t D, qr_dtype dt, const char* who);

#define QR_CUDA_OK(expr)                                                                       \
    do {                                                                                       \
        cudaError_t e__ = (expr);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return qr::fail(QR_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));     \
    } while (0)

// every kernel launch of the library passes through QR_LAUNCH_OK: qr_launch_count() reports how many there were
void count_launch();

#define QR_LAUNCH_OK(name)                                                                     \
    do {                                                                                       \
        qr::count_launch();                                                                    \
        cudaError_t e__ = cudaGetLastError();                                                  \
        if (e__ != cudaSuccess)                                                                \
            return qr::fail(QR_ERR_CUDA, "launch of %s failed: %s", name, cudaGetErrorString(e__)); \
    } while (0)

// SMs of the current device (148 on B200)
int sm_count();

// 32-bit integer mixer (the public-domain "lowbias32" constants): shared-memory hash sets of Gaussian ids
__host__ __device__ __forceinline__ uint32_t hash32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

// qr_bin.cu: inclusive prefix sum of uint32 counts (three launches); sums = scan_blocks(N) uint64 of scratch
int64_t scan_blocks(int64_t N);
int launch_inclusive_scan_u32(const uint32_t* in, int64_t N, uint64_t* out, uint64_t* sums, cudaStream_t st);

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace qr
