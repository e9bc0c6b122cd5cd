/* The C ABI of libfdham used from plain C99 (tests/test_abi.py compiles and runs this file): the
 * header must compile as C, the library must link without any C++ or torch symbol, and argument
 * errors must come back as fd_status values.  No GPU is needed: a valid fd_create returns FD_OK on a
 * GPU box and FD_ERR_CUDA elsewhere (there is no CPU fallback). */
#include <stdio.h>
#include <string.h>

#include "fdham.h"

int main(void)
{
    const int32_t shape[3] = { 8, 8, 8 }, bad_shape[3] = { 8, 0, 8 };
    const double h[3] = { 0.4, 0.4, 0.4 };
    const int32_t bc[3] = { FD_BC_PERIODIC, FD_BC_ZERO, FD_BC_PERIODIC };
    fd_plan *plan = NULL;
    int32_t info[8];
    int rc;

    if (strcmp(fd_strerror(FD_OK), "success") != 0) return 1;
    if (fd_create(&plan, bad_shape, h, 3, bc, NULL, FD_F64, 0) != FD_ERR_INVALID || plan) return 2;
    if (fd_create(&plan, shape, h, 9, bc, NULL, FD_F64, 0) != FD_ERR_INVALID) return 3;
    if (fd_apply_kinetic(NULL, NULL, NULL, 1, NULL) != FD_ERR_INVALID) return 4;
    if (fd_expect_workspace_bytes(NULL, 1) != FD_ERR_INVALID) return 5;
    if (fd_restrict(NULL, bc, 1, NULL, NULL, 1, NULL) != FD_ERR_INVALID) return 6;
    if (fd_paw_nproj_total(NULL) != FD_ERR_INVALID) return 7;
    if (fd_destroy(NULL) != FD_OK || fd_paw_destroy(NULL) != FD_OK || fd_workspace_destroy(NULL) != FD_OK)
        return 8;
    /* the no-allocation entry point: usable from C, its limit is a compile-time constant, its own
     * status code has a message; a single-precision caller passes float * as v_eff without a cast */
    if (fd_apply_hamiltonian_expect_static(NULL, NULL, NULL, NULL, NULL, NULL, 1, NULL) != FD_ERR_INVALID)
        return 12;
    if (FD_STATIC_SCRATCH_BYTES != 4 * 1024 * 1024 || !strstr(fd_strerror(FD_ERR_SCRATCH), "scratch"))
        return 13;
    {
        const float *v32 = NULL;
        if (fd_apply_hamiltonian(NULL, NULL, v32, NULL, 1, NULL) != FD_ERR_INVALID) return 14;
    }
    if (fd_mg_get_info(NULL, NULL) != FD_ERR_INVALID) return 15;
    rc = fd_create(&plan, shape, h, 3, bc, NULL, FD_C128, 0);
    if (rc == FD_OK) {
        if (fd_plan_get_info(plan, info) != FD_OK || info[0] != 8 || info[3] != 3 || info[4] != FD_C128)
            return 9;
        if (fd_apply_kinetic(plan, NULL, NULL, 0, NULL) != FD_OK) return 10; /* nbands == 0: no-op */
        fd_destroy(plan);
        printf("c_abi_check: device present, plan created\n");
    } else if (rc == FD_ERR_CUDA) {
        printf("c_abi_check: no usable CUDA device, fd_create says: %s\n", fd_strerror(rc));
    } else {
        return 11;
    }
    return 0;
}
