// placeholder until the structured solver lands (next commit)
#include "pinmpc_common.cuh"
size_t pinmpc_srb_smem_bytes(int, int) { return 0; }
int pinmpc_launch_solve_srb(pinmpc_ctx *h, cudaStream_t)
{
    snprintf(h->err, sizeof h->err, "structured solver not built");
    return -1;
}
