"""Env sharding for N GPUs: contiguous env ranges, no collective on the data path.

Environments are independent, the layout and the SDF bank are replicated, all state is per env,
and the Philox counters use the GLOBAL env id, so rank r creates its context with
`env_id_base = shard_range(E, world, r)[0]` and its slice of every [E, ...] array; the concatenation of
the ranks' outputs is bit-identical to the single-GPU run.
"""


def shard_range(n_envs, world_size, rank):
    """-> (first_env, count) of `rank`; the first n_envs % world_size ranks get one extra env."""
    if not (0 <= rank < world_size) or n_envs < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(int(n_envs), int(world_size))
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def shard_inputs(inputs, first_env, count):
    """Slices every per-env array of a step-input dict."""
    return {k: v[first_env:first_env + count] for k, v in inputs.items()}
