// qr_api.cu -- version, error string and argument checks shared by every C-ABI entry point (include/qr.h).
#include "qr_common.cuh"

namespace qr {

char* err_buf()
{
    static thread_local char buf[512] = {0};
    return buf;
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

}  // namespace qr

extern "C" int qr_version(void) { return QR_VERSION; }

extern "C" const char* qr_last_error(void) { return qr::err_buf(); }

extern "C" int32_t qr_num_tiles(const qr_camera* cam)
{
    if (!cam || cam->width < 1 || cam->height < 1) return 0;
    return ((cam->width + qr::kTile - 1) / qr::kTile) * ((cam->height + qr::kTile - 1) / qr::kTile);
}
