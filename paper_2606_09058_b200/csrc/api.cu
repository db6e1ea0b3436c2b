// api.cu -- status strings, version, launch counter (C-ABI).
#include "nao_internal.cuh"


NAO_EXPORT const char *nao_status_string(int status) {
    switch (status) {
        case NAO_OK: return "ok";
        case NAO_ERR_WORKSPACE: return "workspace too small";
        case NAO_ERR_CUDA: return "CUDA runtime or launch error";
        case NAO_ERR_ELECTRONS: return "n_electrons outside (0, sum of weights * n) or kT <= 0";
        case NAO_ERR_UNSUPPORTED: return "unsupported combination of arguments";
        default: return status < 0 ? "invalid argument (index = -status)" : "unknown status";
    }
}
NAO_EXPORT const char *nao_version(void) { return "nao-b200 0.1 (sm_100a)"; }
NAO_EXPORT long nao_launch_count(void) { return nao::g_launch_count; }
