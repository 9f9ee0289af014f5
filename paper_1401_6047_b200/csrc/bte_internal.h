// bte_internal.h -- what the translation units of libbte_b200 share besides include/bte.h.  Not installed, not exported
// (the library is built with -fvisibility=hidden; only the functions of include/bte.h carry BTE_API).
#pragma once

// sets the thread-local text behind bte_last_error()
void bte_internal_set_error(const char* text);
