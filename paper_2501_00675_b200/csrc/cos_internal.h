// cos_internal.h -- accessors shared by the translation units of libcos_b200.so (not part of include/cos.h).
#pragma once
#include "../../include/cos.h"
#ifdef __cplusplus
extern "C" {
#endif
int cos_internal_device(const cos_ctx* ctx);      /* CUDA device ordinal of the ctx */
void* cos_internal_stream(const cos_ctx* ctx);    /* cudaStream_t of the ctx */
#ifdef __cplusplus
}
#endif
