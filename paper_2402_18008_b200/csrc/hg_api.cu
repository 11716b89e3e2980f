// hg_api.cu -- status strings and build information of libhg.
#include "hg_host.h"

#define HG_VERSION_NUMBER 100   /* 0.1.0 */

extern "C" const char* hg_status_string(int status)
{
    switch (status) {
        case HG_OK:              return "HG_OK";
        case HG_ERR_INVALID_ARG: return "HG_ERR_INVALID_ARG: null pointer, negative size or unknown enum value";
        case HG_ERR_ALIGNMENT:   return "HG_ERR_ALIGNMENT: a base pointer is not sufficiently aligned";
        case HG_ERR_CUDA:        return "HG_ERR_CUDA: a CUDA runtime call or kernel launch failed";
        case HG_ERR_WORKSPACE:   return "HG_ERR_WORKSPACE: workspace smaller than hg_ransac_workspace_bytes()";
        case HG_ERR_TOO_LARGE:   return "HG_ERR_TOO_LARGE: size beyond the fixed capacity of a no-allocation entry point";
        default:                 return "unknown hg status";
    }
}

extern "C" int hg_version(void) { return HG_VERSION_NUMBER; }

// 100 for sm_100a: the only architecture this library is written for.
extern "C" int hg_built_for_sm(void) { return 100; }
