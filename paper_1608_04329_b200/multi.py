"""Multi-GPU plumbing: one process per GPU, two modes.
  * independent chains, one per rank (seed + rank): no data-path collective; torch.distributed only reduces the
    timing and gathers the draws of all chains (cross-chain convergence diagnostics);
  * ONE chain with the rows of X sharded over the ranks (`sharded_init`, `sharded_sweeps`): one all-reduce of the
    p x p Gram at init and one all-reduce of X^T z (p doubles) per sweep, issued on the chain's own stream.
Nothing here touches the sampler's arithmetic; it works on any backend (nccl on GPUs, gloo in the CPU tests)."""
import torch
import torch.distributed as dist


def world():
    """(rank, world_size) of the default process group, (0, 1) when none is initialised."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def chain_seed(base_seed, rank):
    """Philox seed of the chain on `rank`: distinct keys give independent streams (counter-based RNG)."""
    return (int(base_seed) + int(rank)) & 0xFFFFFFFFFFFFFFFF


def max_over_ranks(value, device="cpu"):
    """Device-timed milliseconds -> the maximum over ranks (the job is as slow as its slowest rank)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world()[1] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank, ms_max):
    """Whole-job throughput: units all ranks processed / the slowest rank's time."""
    return world()[1] * units_per_rank / (ms_max * 1e-3)


def gather_draws(draws):
    """draws: tensor [n_iter, d] of this rank's chain -> tensor [world, n_iter, d] on every rank."""
    draws = draws.contiguous()
    _, ws = world()
    if ws == 1:
        return draws.unsqueeze(0)
    out = [torch.empty_like(draws) for _ in range(ws)]
    dist.all_gather(out, draws)
    return torch.stack(out)


def split_rhat(chains):
    """Split-R-hat of Gelman et al. per coordinate; chains: [m, n, d] (m chains of n draws).  Each chain is
    split in two halves, so the statistic also detects a drifting single chain."""
    m, n, d = chains.shape
    h = n // 2
    x = torch.cat([chains[:, :h], chains[:, h:2 * h]], dim=0).to(torch.float64)     # [2m, h, d]
    means = x.mean(dim=1)
    W = x.var(dim=1, unbiased=True).mean(dim=0)
    B = h * means.var(dim=0, unbiased=True)
    var_plus = (h - 1) / h * W + B / h
    return torch.sqrt(var_plus / W)


# ---- row-sharded chain (include/hsp.h "Row-sharded chains"): the driver loop, on any chain object that offers
# sweep_prepare(n) / sweep_begin() / sweep_end(), xtz_tensor() and gram_tensor() (HorseshoeProbit created with
# row_offset=...; the CPU tests drive an oracle-backed stand-in through the same loop).

def shard_rows(N, rank, world_size):
    """Rows [r0, r1) of rank `rank`: contiguous, sizes differ by at most one row."""
    base, rem = divmod(int(N), int(world_size))
    r0 = rank * base + min(rank, rem)
    return r0, r0 + base + (1 if rank < rem else 0)


def _check_stream(chain):
    """The collective is ordered against the chain's kernels only if both are enqueued on the SAME stream: the chain
    must have been created on an explicit stream and that stream must be torch's current stream here.  (A chain created
    without a stream runs on a private stream of the library: the all-reduce would race with reduce_partials and the
    beta draw.)  Chains that are not CUDA chains (the CPU stand-in of the gloo tests) have no stream_handle."""
    handle = getattr(chain, "stream_handle", None)
    if handle is None:
        return
    g = chain.xtz_tensor()
    if not g.is_cuda:
        return
    cur = torch.cuda.current_stream(g.device).cuda_stream
    if handle() == 0 or handle() != cur:
        raise RuntimeError("row-sharded chain: create the chain with stream=<torch stream> and call sharded_init / "
                           "sharded_sweeps inside `with torch.cuda.stream(<that stream>)`; chain stream = %#x, current = %#x"
                           % (handle(), cur))


def sharded_init(chain, group=None):
    """Sum the per-shard Gram matrices in place, once (p*p doubles)."""
    _check_stream(chain)
    if world()[1] > 1:
        dist.all_reduce(chain.gram_tensor(), op=dist.ReduceOp.SUM, group=group)


def sharded_sweeps(chain, n_iter, group=None):
    """n_iter sweeps of a row-sharded chain: per sweep one all-reduce of X^T z (p doubles) between the local pass
    and the beta draw.  Everything is enqueued on the current stream; there is no host synchronisation."""
    _check_stream(chain)
    chain.sweep_prepare(n_iter)
    g = chain.xtz_tensor()
    ws = world()[1]
    for _ in range(n_iter):
        chain.sweep_begin()
        if ws > 1:
            dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)
        chain.sweep_end()
