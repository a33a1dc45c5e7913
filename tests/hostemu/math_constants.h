// math_constants.h -- TEST INFRASTRUCTURE: the constants of the CUDA header of the same name that libvr uses
// (host emulation, see cuda_runtime.h in this directory).
#pragma once
#define CUDART_INF_F __builtin_huge_valf()
#define CUDART_NAN_F __builtin_nanf("")
