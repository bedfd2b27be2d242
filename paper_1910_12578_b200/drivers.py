"""Harness-level SDC drivers (SURVEY 8(c) S5 "Driver"; Eq. (2) with R = 0).

The library exports the steps of the path (ghost fill, <A(U)>, node update, CFL); the node loop that strings
them into one time step is not part of the C ABI.  Everything here is a sequence of library calls through
binding.Context -- no arithmetic on the state happens in Python.
"""


def sdc_step_2nd(ctx, U, U1, A0, A1, dt, stream=None):
    """One 2-node, 2-iteration SDC step (trapezoid, R = 0) from library calls only.
    U: state with interior valid (ghosts are filled here); result left in U (interior).
    U1, A0, A1: caller-owned work buffers (U1 like U, A0/A1 interior-sized)."""
    w = [0.5 * dt, 0.5 * dt]
    ctx.fill_ghosts(U, stream)
    # iteration 1: every node carries A(U^n): A0 = A(U), U1 = U + dt*A0 (fused)
    ctx.advance_A_update(U, A0, U1, dt, A0, [A0, A0], w, stream)
    ctx.fill_ghosts(U1, stream)
    ctx.advance_A(U1, A1, stream)
    # iteration 2: node 0 unchanged, integral from iteration-1 values (trapezoid)
    ctx.sdc_update(U, U, dt, A0, A0, [A0, A1], w, stream)


# Gauss-Lobatto node-to-node quadrature weights (fractions of dt) for M = 2 (trapezoid) and M = 3 (Simpson),
# PAPER.md L44; rows m = 0..M-2, columns j = 0..M-1 (Q17).
_SDC_WEIGHTS = {2: [[1.0 / 2.0, 1.0 / 2.0]],
                3: [[5.0 / 24.0, 8.0 / 24.0, -1.0 / 24.0], [-1.0 / 24.0, 8.0 / 24.0, 5.0 / 24.0]]}


def sdc_step_nodes(ctx, U, dt, M=3, K=4, stream=None):
    """One SDC step with M Gauss-Lobatto nodes and K iterations (Eq. (2) of the paper, R = 0) from library
    calls only: cst_fill_ghosts, cst_advance_A, cst_sdc_update.  U: state with interior valid; result left
    in U (interior).  Work buffers (M - 1 states, 2 M - 1 A arrays) are torch allocations made here."""
    import torch
    wt = _SDC_WEIGHTS[M]
    dtm = dt / (M - 1)
    ashape = (U.shape[0], U.shape[1], U.shape[2] - 8, U.shape[3] - 8, U.shape[4] - 8)
    new_A = lambda: torch.empty(ashape, dtype=U.dtype, device=U.device)
    ctx.fill_ghosts(U, stream)
    A0 = new_A()
    ctx.advance_A(U, A0, stream)
    A_old = [A0] * M
    A_buf = [[new_A() for _ in range(M - 1)] for _ in range(2)]
    U_nodes = [U] + [torch.empty_like(U) for _ in range(M - 1)]
    for k in range(K):
        A_new = [A0]
        for m in range(M - 1):
            ctx.sdc_update(U_nodes[m + 1], U_nodes[m], dtm, A_new[m], A_old[m], A_old,
                           [w * dt for w in wt[m]], stream)
            if k == K - 1 and m == M - 2:
                break
            ctx.fill_ghosts(U_nodes[m + 1], stream)
            ctx.advance_A(U_nodes[m + 1], A_buf[k % 2][m], stream)
            A_new.append(A_buf[k % 2][m])
        A_old = A_new
    if M > 1:
        U.copy_(U_nodes[M - 1])


def sdc_step_nodes_react(ctx, U, dt, M=3, K=4, stream=None):
    """One SDC step of Eq. (2) with R != 0: M Gauss-Lobatto nodes, K iterations, A explicit,
    R implicit (cst_sdc_update_react; needs ctx.set_reactions).  Library calls only.  U: state with interior valid;
    result left in U (interior)."""
    import torch
    wt = _SDC_WEIGHTS[M]
    dtm = dt / (M - 1)
    ashape = (U.shape[0], U.shape[1], U.shape[2] - 8, U.shape[3] - 8, U.shape[4] - 8)
    new_A = lambda: torch.empty(ashape, dtype=U.dtype, device=U.device)
    ctx.fill_ghosts(U, stream)
    A0, R0 = new_A(), new_A()
    ctx.advance_A(U, A0, stream)
    ctx.react_R(U, R0, stream)
    A_old, R_old = [A0] * M, [R0] * M
    A_buf = [[new_A() for _ in range(M - 1)] for _ in range(2)]
    R_buf = [[new_A() for _ in range(M - 1)] for _ in range(2)]
    U_nodes = [U] + [torch.empty_like(U) for _ in range(M - 1)]
    for k in range(K):
        A_new, R_new = [A0], [R0]
        for m in range(M - 1):
            Rn = R_buf[k % 2][m]
            ctx.sdc_update_react(U_nodes[m + 1], U_nodes[m], dtm, A_new[m], A_old[m], R_old[m + 1], A_old, R_old,
                                 [w * dt for w in wt[m]], Rn, stream)
            R_new.append(Rn)
            if k == K - 1 and m == M - 2:
                break
            ctx.fill_ghosts(U_nodes[m + 1], stream)
            ctx.advance_A(U_nodes[m + 1], A_buf[k % 2][m], stream)
            A_new.append(A_buf[k % 2][m])
        A_old, R_old = A_new, R_new
    if M > 1:
        U.copy_(U_nodes[M - 1])
