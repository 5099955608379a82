// errors.hpp -- the thread-local status / message behind cans_last_status() and cans_last_error(), for the translation units
// other than cans_poisson.cu (which owns the storage).  Each returns the code it recorded.
#pragma once
#include <cuda_runtime.h>

namespace cans {

void report_ok();                                             // entry points start with this: status CANS_OK
int report_failure(int code, const char* message);
int report_cuda_failure(cudaError_t e, const char* where);   // CANS_ERR_CUDA, "<where>: <CUDA error string>"

}  // namespace cans
