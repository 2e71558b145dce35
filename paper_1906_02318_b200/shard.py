"""Host-side plumbing of the sharded tick: which candidate range a rank owns,
and the collective that exchanges the 24-byte partials.  No arithmetic of the method lives here: the
rollout, the per-shard argmin and the final reduction + decode run in the kernels
(mpmi_shard_step / mpmi_shard_finalize)."""
import torch

KEY_INDEX_BITS = 30


def shard_plan(N, include_user, world, rank):
    """Global candidate indices [begin, begin + count) owned by `rank`: N sampled candidates split
    as evenly as possible, the injected user input (index N) appended to the last rank."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, extra = divmod(int(N), world)
    begin = rank * base + min(rank, extra)
    count = base + (1 if rank < extra else 0)
    if rank == world - 1 and include_user:
        count += 1
    return begin, count


def gather_partials(partial, world, group=None):
    """all-gather of one (3,) int64 partial per rank -> (world*3,) int64 on every rank.
    NCCL over NVLink on GPUs (24 bytes per rank: latency-bound), gloo on CPU in the tests."""
    out = torch.empty(3 * world, dtype=torch.int64, device=partial.device)
    torch.distributed.all_gather_into_tensor(out, partial.contiguous(), group=group)
    return out


def decode_key(key):
    """(unsafe_flag, primary, index) of a packed selection key (layout: DESIGN.md section 5)."""
    key = int(key)
    return (key >> 62) & 1, (key >> KEY_INDEX_BITS) & 0xFFFFFFFF, key & ((1 << KEY_INDEX_BITS) - 1)
