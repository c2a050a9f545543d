// nd_internal.h -- private helpers shared by the translation units of libnd_moc.so (never installed).
#ifndef ND_INTERNAL_H
#define ND_INTERNAL_H
#include "nd.h"

// Records `msg` as the calling thread's last error and returns `s` (so callers can `return nd_fail(...)`).
nd_status nd_fail(nd_status s, const char* msg);

#endif
