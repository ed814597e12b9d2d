"""The annealing loop of PAPER.md L55-L63 (steps 1-5), written once against the call names of
include/pa.h so that the same driver runs the CPU oracle (oracle.pa_oracle.Oracle) and the CUDA
library (paper_1703_03676_b200.pa.Population).  Holds no arithmetic of the method."""


def run_fixed(pop, betas, theta, hist=False, on_step=None):
    """betas[0] = beta_0; for every later beta: resample, theta sweeps, measure."""
    out = [pop.observables(betas[0])]
    if hist:
        pop.hist_accumulate(betas[0])
    for i in range(1, len(betas)):
        pop.resample(betas[i - 1], betas[i])
        pop.sweep(betas[i], theta)
        out.append(pop.observables(betas[i]))
        if hist:
            pop.hist_accumulate(betas[i])
        if on_step is not None:
            on_step(i, pop)
    return out


def run_adaptive(pop, beta0, beta_f, theta, target, hist=False, max_steps=100000, on_step=None):
    beta = beta0
    betas = [beta]
    out = [pop.observables(beta)]
    if hist:
        pop.hist_accumulate(beta)
    i = 0
    while beta < beta_f and i < max_steps:
        i += 1
        dbeta = pop.adapt_dbeta(target, beta, beta_f)
        new = beta_f if beta + dbeta >= beta_f else beta + dbeta
        pop.resample(beta, new)
        pop.sweep(new, theta)
        beta = new
        betas.append(beta)
        out.append(pop.observables(beta))
        if hist:
            pop.hist_accumulate(beta)
        if on_step is not None:
            on_step(i, pop)
    return betas, out
