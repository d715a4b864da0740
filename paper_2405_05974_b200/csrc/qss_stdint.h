// Internal: fixed-width integer types for sources that are also compiled at run time by NVRTC (which has no <stdint.h>).
#ifndef QSS_STDINT_H
#define QSS_STDINT_H
#ifdef __CUDACC_RTC__
typedef signed int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
#else
#include <stdint.h>
#endif
#endif
