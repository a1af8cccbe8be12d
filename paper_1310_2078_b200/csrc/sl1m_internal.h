// sl1m_internal.h -- shared between the translation units of libsl1m.so; not part of the ABI.
#pragma once

// Records `msg` as the thread's sl1m_last_error() text and returns `st` (defined in sl1m.cu).
int sl1m_fail(int st, const char *msg);
