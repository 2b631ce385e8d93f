/* tests/host/simt/simt_switch.S - TEST INFRASTRUCTURE: the fibre switch of cuda_runtime.h on x86-64 (System V ABI).
   void nb_simt_switch(void** save_sp, void* load_sp): push the callee-saved registers, store the stack pointer in *save_sp,
   take load_sp as the stack pointer, pop the callee-saved registers found there, return to the address that follows them. */
#if defined(__x86_64__)
    .text
    .globl nb_simt_switch
    .type nb_simt_switch, @function
nb_simt_switch:
    pushq %rbp
    pushq %rbx
    pushq %r12
    pushq %r13
    pushq %r14
    pushq %r15
    movq %rsp, (%rdi)
    movq %rsi, %rsp
    popq %r15
    popq %r14
    popq %r13
    popq %r12
    popq %rbx
    popq %rbp
    ret
    .size nb_simt_switch, .-nb_simt_switch
    .section .note.GNU-stack,"",@progbits
#endif
