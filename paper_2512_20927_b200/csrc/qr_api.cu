// qr_api.cu -- version, error string and argument checks shared by every C-ABI entry point (include/qr.h).
#include "qr_common.cuh"
#include "qr_sel.cuh"

#include <atomic>

namespace qr {

char* err_buf()
{
    static thread_local char buf[512] = {0};
    return buf;
}

static std::atomic<long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

int sm_count()
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
        n = 148;
    return n;
}

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err_buf(), 512, fmt, ap);
    va_end(ap);
    return code;
}

int check_cam(const qr_camera* cam)
{
    if (!cam) return fail(QR_ERR_NULL_POINTER, "camera is NULL");
    if (cam->width < 1 || cam->height < 1)
        return fail(QR_ERR_INVALID_ARG, "zero-area image %d x %d (SPEC.md:143)", cam->width, cam->height);
    if (!(cam->znear > 0.0f)) return fail(QR_ERR_INVALID_ARG, "znear must be > 0");
    if (!(cam->fx > 0.0f) || !(cam->fy > 0.0f)) return fail(QR_ERR_INVALID_ARG, "focal lengths must be > 0");
    const int64_t tx = (cam->width + kTile - 1) / kTile, ty = (cam->height + kTile - 1) / kTile;
    if (tx * ty >= (int64_t(1) << 24)) return fail(QR_ERR_UNSUPPORTED, "more than 2^24 tiles");
    return QR_OK;
}

int check_feat(int32_t D, qr_dtype dt, const char* who)
{
    if (D < 1) return fail(QR_ERR_INVALID_ARG, "%s: D = %d < 1", who, D);
    if (D > QR_MAX_D) return fail(QR_ERR_UNSUPPORTED, "%s: D = %d > QR_MAX_D", who, D);
    if (dt != QR_F32 && dt != QR_F16) return fail(QR_ERR_INVALID_ARG, "%s: unknown feature dtype %d", who, (int)dt);
    if (dt == QR_F16 && D % 8 != 0) return fail(QR_ERR_UNSUPPORTED, "%s: fp16 features need D %% 8 == 0", who);
    if (dt == QR_F32 && D % 4 != 0 && D > 128)
        return fail(QR_ERR_UNSUPPORTED, "%s: D %% 4 != 0 is only supported for D <= 128", who);
    return QR_OK;
}

// sums over the half-tile headers the walk left in a forward workspace (qr_sel.cuh)
__global__ void forward_stats_kernel(const int32_t* __restrict__ hdr, int num_half, long long* __restrict__ out)
{
    long long ent = 0, uni = 0, cons = 0, ev = 0, cyc = 0, big = 0;
    for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < num_half; h += gridDim.x * blockDim.x) {
        const int32_t* d = hdr + (size_t)h * kHdrWords;
        ent += (long long)d[0] + d[1] + d[2] + d[3];
        uni += d[4]; cons += d[6]; ev += d[7]; cyc += d[8]; big += d[4] > 64 ? 1 : 0;
    }
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 0), (unsigned long long)ent);
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 1), (unsigned long long)uni);
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 2), (unsigned long long)cons);
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 3), (unsigned long long)ev * 32ull);
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 4), (unsigned long long)cyc);
    atomicAdd(reinterpret_cast<unsigned long long*>(out + 5), (unsigned long long)big);
}

}  // namespace qr

extern "C" long long qr_launch_count(void) { return qr::g_launches.load(std::memory_order_relaxed); }

extern "C" int qr_forward_stats(const qr_camera* cam, int32_t K, const void* fwd_ws, size_t fwd_ws_bytes, int64_t* stats, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1 || K > QR_MAX_K) return fail(QR_ERR_INVALID_ARG, "qr_forward_stats: K out of range");
    if (!fwd_ws || !stats) return fail(QR_ERR_NULL_POINTER, "qr_forward_stats: NULL argument");
    const Cam c = make_cam(cam);
    const WsLayout wl = ws_layout(c, K);
    if (fwd_ws_bytes < wl.total) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_forward_stats: workspace %zu < %zu bytes", fwd_ws_bytes, wl.total);
    const SelLists sl = sel_view(wl.sel, const_cast<void*>(fwd_ws));
    cudaStream_t st = (cudaStream_t)stream;
    QR_CUDA_OK(cudaMemsetAsync(stats, 0, 8 * sizeof(int64_t), st));
    const int nh = c.tiles_x * c.tiles_y * 2;
    forward_stats_kernel<<<(nh + 255) / 256, 256, 0, st>>>(sl.hdr, nh, reinterpret_cast<long long*>(stats));
    QR_LAUNCH_OK("forward_stats_kernel");
    return QR_OK;
}

extern "C" int qr_version(void) { return QR_VERSION; }

extern "C" const char* qr_last_error(void) { return qr::err_buf(); }

extern "C" int32_t qr_num_tiles(const qr_camera* cam)
{
    if (!cam || cam->width < 1 || cam->height < 1) return 0;
    return ((cam->width + qr::kTile - 1) / qr::kTile) * ((cam->height + qr::kTile - 1) / qr::kTile);
}
