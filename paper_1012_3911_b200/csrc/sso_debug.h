/*
 * sso_debug.h -- test scaffolding, NOT part of the public C ABI of include/sso.h.
 *
 * Host-only introspection of the plan builder (no GPU needed; tests/test_abi.py checks the permuted table layout with
 * it): for a line of n points, pos_freq[p] = frequency index held at position p after the decimation-in-frequency
 * stages, and slot_nat[s] = natural index stored at slot s of the permuted table layout.  Both are host int[n].
 * Returns SSO_OK, or SSO_ERR_INVALID for an n that is not a supported power of two.
 */
#ifndef SSO_DEBUG_H
#define SSO_DEBUG_H
#ifdef __cplusplus
extern "C" {
#endif
int sso_debug_layout(int n, int *pos_freq, int *slot_nat);
#ifdef __cplusplus
}
#endif
#endif
