// wslda.cu -- the single translation unit of libwslda (C-ABI in include/wslda.h).
// Build: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -shared -Xcompiler -fPIC wslda.cu -o libwslda.so
#include "step.cuh"
