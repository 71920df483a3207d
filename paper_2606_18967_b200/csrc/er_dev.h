/* er_dev.h -- entry points that exist ONLY in the development build of the library (liber_b200_dev.so, compiled with
 * -DER_DEV by `python -m paper_2606_18967_b200.build --dev`).  They select the work partition / launch mode / kernel
 * variant the plan would otherwise choose by itself, so that the tests can compare every one of them against the
 * oracle.  They set process-global state and are NOT part of the C ABI of include/er.h: the shipped liber_b200.so
 * neither exports them nor contains the variables behind them (tests/test_abi.py checks its export list). */
#ifndef ER_DEV_H_
#define ER_DEV_H_
#ifdef __cplusplus
extern "C" {
#endif

/* key 1: number of CTAs of the W4A16 GEMM (0 = one per SM); 3: programmatic dependent launch (0/1);
 * 4: tile split (0/1); 5: thread-block-cluster mode (0/1); 6: M <= 8 through the warp-level-MMA kernel (0/1);
 * 7: the pre-scaled large-batch kernel (development library only): 0 never (default, as in the shipped library), 1 for
 * M > 64, 2 for every M > 16; 8: M > 64 through the 128-row kernel (1, default) or in chunks of 64 rows (0). */
int er_dev_gemm_tuning(int key, int value);
/* CTAs per sequence of er_spec_verify: 0 = automatic, or 1 / 2 / 4 / 8.  16 / 17: the shared-memory ring kernel
 * where it applies (default) / the register-path kernel for every input. */
int er_dev_verify_cluster(int cluster);

#ifdef __cplusplus
}
#endif
#endif /* ER_DEV_H_ */
