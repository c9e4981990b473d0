// api_errors.h — the library's one error channel, shared by every translation unit that implements C-ABI calls.
// The status codes are dash_hash4d_status; the message is what dash_hash4d_last_error() returns (thread-local).
// Defined in hash4d_api.cu.
#pragma once
#include <cuda_runtime.h>

namespace dash {

// Store a printf-style message for dash_hash4d_last_error() and return `code` (a non-OK dash_hash4d_status).
int api_fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
// DASH_HASH4D_CUDA_ERROR with "<what>: <cudaGetErrorString(e)>".
int api_cuda_fail(cudaError_t e, const char* what);
// Clear the message and return DASH_HASH4D_OK.
int api_ok();

}  // namespace dash
