"""Row sharding for N > 1 GPUs: every row is independent, so rank k of N takes a
contiguous row range and there is no data-path collective; only throughput bookkeeping is reduced."""
from typing import Tuple


def shard_rows(n: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of rank's contiguous shard; shards differ by at most two rows and have even begin offsets
    (keeps 16-byte alignment of fp64 arrays for the vector path)."""
    if world <= 0 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    pairs = n // 2
    base, rem = divmod(pairs, world)
    begin = 2 * (rank * base + min(rank, rem))
    end = 2 * ((rank + 1) * base + min(rank + 1, rem))
    if rank == world - 1:
        end = n
    return begin, end
