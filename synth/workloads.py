"""Region generators and mutators (torch, device-agnostic; seeded; no method arithmetic).

All generators return flat ``torch.uint8`` tensors on ``device`` (views of the typed
data), because the checkpoint path treats every region as bytes (PAPER.md:L261
"compares opaque regions against shadows"; BASELINE.json config 3 "bitwise compare").
Page choices are "first k of a seeded randperm, sorted".
"""
import math
from dataclasses import dataclass

import torch

__all__ = [
    "gen", "choose_pages", "raw_region", "mutate_byte_flips", "kv_cache_region", "kv_decode_step",
    "lora_region", "lora_update", "bf16_normal_region", "sparse_xor_flips", "toggle_flips", "all_dirty_flips",
    "RecoveryEpoch", "recovery_epochs", "worker_mutation_pages", "C5A_REGIONS",
]


def gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def choose_pages(n_pages: int, k: int, g: torch.Generator) -> torch.Tensor:
    """k distinct page indices, ascending (int64, on g's device)."""
    perm = torch.randperm(n_pages, generator=g, device=g.device)
    return torch.sort(perm[:k]).values


# ------------------------------------------------------------------ C1: raw bytes --

def raw_region(n_bytes: int, seed: int, device) -> torch.Tensor:
    """Uniform random bytes (config 1 / 5)."""
    g = gen(seed, device)
    out = torch.empty(n_bytes, dtype=torch.uint8, device=device)
    step = 1 << 28
    for o in range(0, n_bytes, step):
        n = min(step, n_bytes - o)
        out[o:o + n] = torch.randint(0, 256, (n,), dtype=torch.uint8, generator=g, device=device)
    return out


def mutate_byte_flips(region: torch.Tensor, page_bytes: int, ratio: float, seed: int,
                      max_flips: int = 8) -> torch.Tensor:
    """Config 1: ceil(ratio*n_pages) pages, each with 1..max_flips XOR flips (non-zero mask)
    at distinct offsets; chosen page #0 includes offset 0, #1 offset page_bytes-1, #2 both.
    Returns the ascending page list (int64, cpu).  Mutates ``region`` in place."""
    n = region.numel()
    n_pages = (n + page_bytes - 1) // page_bytes
    k = max(1, math.ceil(ratio * n_pages))
    g = gen(seed, "cpu")
    pages = choose_pages(n_pages, k, g)
    offs_all, mask_all = [], []
    for j, p in enumerate(pages.tolist()):
        plen = min(page_bytes, n - p * page_bytes)
        m = int(torch.randint(1, max_flips + 1, (1,), generator=g))
        m = min(m, plen)
        offs = torch.randperm(plen, generator=g)[:m]
        if j == 0:
            offs[0] = 0
        if j == 1:
            offs[0] = plen - 1
        if j == 2:
            offs = torch.unique(torch.cat([offs, torch.tensor([0, plen - 1])]))
        offs = torch.unique(offs)
        masks = torch.randint(1, 256, (offs.numel(),), generator=g, dtype=torch.int64).to(torch.uint8)
        offs_all.append(offs + p * page_bytes)
        mask_all.append(masks)
    offs = torch.cat(offs_all).to(region.device)
    masks = torch.cat(mask_all).to(region.device)
    region[offs] = region[offs] ^ masks
    return pages


# ------------------------------------------------------------- C2: paged KV cache --

def kv_cache_region(layers: int, blocks: int, seed: int, device, tokens: int = 16, heads: int = 8,
                    dim: int = 128) -> torch.Tensor:
    """[layers][blocks][2 (K,V)][tokens][heads][dim] bf16 normal(0,1) as flat bytes.
    Default block = 2*16*8*128*2 B = 64 KiB (Llama-3-8B-shaped, config 2)."""
    g = gen(seed, device)
    per_layer = blocks * 2 * tokens * heads * dim
    out = torch.empty(layers * per_layer, dtype=torch.bfloat16, device=device)
    for l in range(layers):
        out[l * per_layer:(l + 1) * per_layer] = torch.randn(per_layer, generator=g, device=device,
                                                             dtype=torch.float32).to(torch.bfloat16)
    return out.view(torch.uint8)


def kv_decode_step(region: torch.Tensor, layers: int, blocks: int, n_seqs: int, seed: int,
                   tokens: int = 16, heads: int = 8, dim: int = 128) -> torch.Tensor:
    """One decode step: per layer, each of n_seqs sequences owns a distinct physical block
    and a slot t in [0,tokens); K[t] and V[t] of that block are overwritten with fresh
    normal(0,1).  Returns ascending dirty block (=page) indices (int64, cpu)."""
    dev = region.device
    g = gen(seed, dev)
    kv = region.view(torch.bfloat16).view(layers, blocks, 2, tokens, heads * dim)
    pages = []
    for l in range(layers):
        blk = torch.randperm(blocks, generator=g, device=dev)[:n_seqs]
        slot = torch.randint(0, tokens, (n_seqs,), generator=g, device=dev)
        new = torch.randn(n_seqs, 2, heads * dim, generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
        kv[l, blk, 0, slot] = new[:, 0]
        kv[l, blk, 1, slot] = new[:, 1]
        pages.append(blk.to(torch.int64) + l * blocks)
    return torch.sort(torch.cat(pages)).values.cpu()


# ------------------------------------------------------------------- C3: LoRA ----

def lora_region(layers: int, seed: int, device, rank: int = 16, hidden: int = 4096, projs: int = 4) -> torch.Tensor:
    """rank-r A[r x hidden] ~ normal(0,0.02) and B[hidden x r] = 0 for q,k,v,o in every layer,
    fp32, packed back to back (config 3: 32 layers -> 64 MiB = 1,024 pages of 64 KiB)."""
    g = gen(seed, device)
    per = rank * hidden
    out = torch.zeros(layers * projs * 2 * per, dtype=torch.float32, device=device)
    v = out.view(layers * projs, 2, per)
    v[:, 0] = torch.randn(layers * projs, per, generator=g, device=device) * 0.02
    return out.view(torch.uint8)


def lora_update(region: torch.Tensor, page_bytes: int, ratio: float, seed: int) -> torch.Tensor:
    """Online update: a seeded ratio of pages gets w += 1e-4*normal(0,1) on every element
    (small-magnitude fp32 deltas).  Asserts that each touched page changed in at least one
    bit.  Returns the ascending page list (int64, cpu)."""
    dev = region.device
    n_pages = region.numel() // page_bytes
    k = max(1, math.ceil(ratio * n_pages))
    g = gen(seed, dev)
    pages = choose_pages(n_pages, k, g)
    w = region.view(torch.float32).view(n_pages, page_bytes // 4)
    old = w[pages].clone()
    w[pages] = old + 1e-4 * torch.randn(old.shape, generator=g, device=dev)
    changed = (w[pages].view(torch.int32) != old.view(torch.int32)).any(dim=1)
    assert bool(changed.all()), "lora_update: a touched page did not change bitwise"
    return pages.cpu()


# --------------------------------------------------------- C4: large bf16 region --

def bf16_normal_region(n_bytes: int, seed: int, device, chunk_bytes: int = 1 << 30) -> torch.Tensor:
    """bf16 normal(0,1) bytes generated chunk-wise (config 4)."""
    g = gen(seed, device)
    out = torch.empty(n_bytes, dtype=torch.uint8, device=device)
    for o in range(0, n_bytes, chunk_bytes):
        n = min(chunk_bytes, n_bytes - o)
        out[o:o + n] = torch.randn(n // 2, generator=g, device=device,
                                   dtype=torch.float32).to(torch.bfloat16).view(torch.uint8)
    return out


def sparse_xor_flips(region: torch.Tensor, page_bytes: int, ratio: float, seed: int):
    """ceil(ratio*n_pages) pages (all pages if ratio >= 1), one XOR flip each at a seeded
    uniform offset.  Returns (pages int64 cpu ascending, flat byte offsets on device, masks on
    device) so that ``toggle_flips`` can re-arm the same dirty set."""
    dev = region.device
    n = region.numel()
    n_pages = (n + page_bytes - 1) // page_bytes
    g = gen(seed, dev)
    if ratio >= 1.0:
        pages = torch.arange(n_pages, device=dev)
    else:
        pages = choose_pages(n_pages, max(1, math.ceil(ratio * n_pages)), g)
    plen = torch.clamp(n - pages * page_bytes, max=page_bytes)
    offs = pages * page_bytes + (torch.rand(pages.numel(), generator=g, device=dev, dtype=torch.float64)
                                 * plen).to(torch.int64).clamp_(max=page_bytes - 1)
    offs = torch.minimum(offs, pages * page_bytes + plen - 1)
    masks = torch.randint(1, 256, (pages.numel(),), generator=g, device=dev, dtype=torch.int64).to(torch.uint8)
    toggle_flips(region, offs, masks)
    return pages.cpu(), offs, masks


def toggle_flips(region: torch.Tensor, offs: torch.Tensor, masks: torch.Tensor) -> None:
    """XOR masks into region[offs] (offsets distinct).  Re-applying toggles the same bytes, which
    keeps the dirty set identical once the shadow holds the previous state."""
    step = 1 << 24
    for o in range(0, offs.numel(), step):
        idx = offs[o:o + step]
        region[idx] = region[idx] ^ masks[o:o + step]


# ------------------------------------------------------------- C5a: recovery log --

# (region_id, byte offset in the arena as a fraction of 8, size fraction of 8, page_bytes)
C5A_REGIONS = ((1, 0, 2, 4096), (2, 2, 2, 16384), (3, 4, 4, 65536))


@dataclass
class RecoveryEpoch:
    epoch: int
    region_id: int
    pages: torch.Tensor      # int64 cpu, distinct within the epoch, in log order (ascending)
    payloads: torch.Tensor   # uint8 cpu, len(pages)*page_bytes


def recovery_epochs(arena_bytes: int, n_epochs: int, recs_per_epoch: int, seed: int, forced_repeats: int = 50):
    """Config 5a: epoch e targets region (e mod 3)+1 of the arena split of C5A_REGIONS; pages are
    distinct within an epoch and may repeat across epochs (at least ``forced_repeats`` forced);
    payloads are uniform random bytes.  The log bytes themselves are written by the ORACLE's record
    writer from these, never by the CUDA path."""
    g = gen(seed, "cpu")
    unit = arena_bytes // 8
    last_pages = {}
    out = []
    forced = 0
    for e in range(n_epochs):
        rid, _, size8, P = C5A_REGIONS[e % 3]
        n_pages = size8 * unit // P
        k = min(recs_per_epoch, n_pages)
        pages = torch.randperm(n_pages, generator=g)[:k]
        if rid in last_pages and forced < forced_repeats:
            pages[0] = last_pages[rid][0]
            pages = torch.unique(pages)
            forced += 1
        pages = torch.sort(pages).values
        last_pages[rid] = pages
        payloads = torch.randint(0, 256, (pages.numel() * P,), dtype=torch.uint8, generator=g)
        out.append(RecoveryEpoch(epoch=e + 1, region_id=rid, pages=pages, payloads=payloads))
    return out


# ------------------------------------------------ C5b: persistent-worker mutation --

def worker_mutation_pages(task_no: int, n_pages: int, n_mut: int, seed: int):
    """Closed-form page set of CC_TASK_TEST_MUTATE: page_j = (j*A + h) mod n_pages,
    j < n_mut, with A odd (so pages are distinct when n_pages is a power of two) and
    h = (seed*2654435761 + task_no*40503) mod 2^32.  Byte offset inside the page = (h + j) mod page
    size is applied by the caller.  Returns (pages list, h)."""
    A = 2 * ((seed * 7919 + 12345) % 100000) + 1
    h = (seed * 2654435761 + task_no * 40503) & 0xFFFFFFFF
    return [((j * A + h) % n_pages) for j in range(n_mut)], h


def all_dirty_flips(n_bytes: int, page_bytes: int, seed: int, device):
    """Config 4, 100 % dirty leg: one seeded byte flip in EVERY page (n_bytes a multiple of page_bytes).  Returns
    (offsets int64, masks uint8) for toggle_flips, ascending -- offsets[p] lies in page p."""
    n_pages = n_bytes // page_bytes
    g = gen(seed, device)
    offs = torch.arange(n_pages, device=device) * page_bytes + torch.randint(0, page_bytes, (n_pages,), generator=g, device=device)
    masks = torch.randint(1, 256, (n_pages,), generator=g, device=device, dtype=torch.int64).to(torch.uint8)
    return offs, masks
