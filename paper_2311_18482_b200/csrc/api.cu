// api.cu — context management and status strings of the legs C-ABI.
#include <new>

#include "common.cuh"

extern "C" {

int legs_create(int device, legs_ctx** out) {
  if (!out) return LEGS_ERR_NULL;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return LEGS_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return LEGS_ERR_CUDA;
  if (prop.major != 10) return LEGS_ERR_CUDA;  // built for sm_100a only; no fallback path
  if (cudaSetDevice(device) != cudaSuccess) return LEGS_ERR_CUDA;
  legs_ctx* c = new (std::nothrow) legs_ctx;
  if (!c) return LEGS_ERR_CUDA;
  c->device = device;
  c->num_sms = prop.multiProcessorCount;
  c->last_cuda_error = 0;
  c->launches = 0;
  c->encode_tiled = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &c->encode_tiled, cudaEnableDefault, &qres) != cudaSuccess ||
      qres != cudaDriverEntryPointSuccess || !c->encode_tiled) {
    delete c;
    return LEGS_ERR_CUDA;
  }
  *out = c;
  return LEGS_OK;
}

void legs_destroy(legs_ctx* ctx) { delete ctx; }

const char* legs_status_string(int status) {
  switch (status) {
    case LEGS_OK: return "ok";
    case LEGS_ERR_NULL: return "required pointer is NULL";
    case LEGS_ERR_ALIGN: return "device pointer is not 16-byte aligned";
    case LEGS_ERR_DIM: return "size or dimension out of range";
    case LEGS_ERR_CAPACITY: return "tile instances exceed capacity";
    case LEGS_ERR_WORKSPACE: return "workspace too small";
    case LEGS_ERR_CUDA: return "CUDA runtime error";
    default: return "unknown status";
  }
}

int legs_last_cuda_error(const legs_ctx* ctx) { return ctx ? ctx->last_cuda_error : 0; }
uint64_t legs_launch_count(const legs_ctx* ctx) { return ctx ? ctx->launches : 0; }
int32_t legs_num_sms(const legs_ctx* ctx) { return ctx ? ctx->num_sms : 0; }

}  // extern "C"
