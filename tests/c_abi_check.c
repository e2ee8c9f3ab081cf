/* c_abi_check.c -- proves that include/rna4r.h compiles as plain C (C99) and that the calls which need no GPU
 * behave as the header says.  Built and run by tests/test_abi.py: gcc -std=c99 -Wall -Werror ... -lrna4r. */
#include <stdio.h>
#include <string.h>
#include "rna4r.h"

int main(void)
{
    rna4r_ctx *ctx = NULL;
    if (strncmp(rna4r_version(), "rna4r", 5) != 0) return 1;
    if (strcmp(rna4r_strerror(RNA4R_OK), "ok") != 0) return 2;
    if (rna4r_prepare(1, 0, NULL, &ctx) != RNA4R_ERR_BAD_Q || ctx != NULL) return 3;      /* q outside 2..12 */
    if (rna4r_prepare(8, 0, NULL, NULL) != RNA4R_ERR_NULL) return 4;
    if (rna4r_destroy(NULL) != RNA4R_ERR_CONTEXT) return 5;
    if (rna4r_workspace_bytes(NULL, 10, 1, RNA4R_WS_DEVICE) != 0) return 6;
    if (rna4r_fold(NULL, NULL, 0, NULL, NULL, RNA4R_TABLE_NONE, NULL, 0, NULL) != RNA4R_ERR_CONTEXT) return 7;
    {
        int rc = rna4r_prepare(8, 0, NULL, &ctx);          /* with a B200: OK; without: DEVICE, never a fallback */
        if (rc == RNA4R_OK) {
            if (rna4r_q(ctx) != 8) return 8;
            if (rna4r_workspace_bytes(ctx, 100, 1, RNA4R_WS_DEVICE) == 0) return 9;
            if (rna4r_workspace_bytes(ctx, 100, 1, RNA4R_WS_HOST_STAGING) <= rna4r_workspace_bytes(ctx, 100, 1, RNA4R_WS_DEVICE)) return 10;
            if (rna4r_destroy(ctx) != RNA4R_OK) return 11;
            printf("c_abi_check ok (device)\n");
        } else if (rc == RNA4R_ERR_DEVICE) {
            printf("c_abi_check ok (no device: %s)\n", rna4r_strerror(rc));
        } else {
            return 12;
        }
    }
    return 0;
}
