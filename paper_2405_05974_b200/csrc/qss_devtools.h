// Internal: development aids are compiled in only when the library is built with -DQSS_DEVTOOLS (build.py: QSS_BUILD_DEV=1).
// The release library reads three environment variables: QSS_VARIANT, QSS_JIT (kernel selection, include/qss.h) and
// QSS_CACHE / QSS_CACHE_DIR (on-disk cache of run-time compiled images); QSS_CS_GLOBAL is kept as a test knob.
#ifndef QSS_DEVTOOLS_H
#define QSS_DEVTOOLS_H
#include <cstdlib>

inline const char *qss_devenv(const char *name) {
#ifdef QSS_DEVTOOLS
    return std::getenv(name);
#else
    (void)name;
    return nullptr;
#endif
}

#endif
