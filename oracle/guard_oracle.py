"""CPU ORACLE of NEXT-3: MGTR accounting and the endpoint-capacity guard. TEST INFRASTRUCTURE
ONLY; plain Python, shares no code with the product.

MGTR — PAPER L110-114: MGTR = sum_e bytes(route_e) / sum_e bytes(FP32_e) over the recorded route events;
"FP32 fallback events and FP32-sensitive tensors count as FP32 bytes, while admitted low-bit tensor portions
count according to the selected low-bit representation"; the denominator replays the same events as FP32.
Readings: an event = (numel, route code, mode); bytes(L) = numel * bits(mode) / 8 + scale_bytes (the per-tensor
mean-absolute scale, L211), bits(G-Binary) = 1, bits(G-Ternary) = log2(3) (reading #14; a parameter);
bytes(F) = bytes(P) = 4 * numel.

Guard — PAPER L273: "admits a candidate low-bit bucket only when the estimated hierarchical-reducer time is
lower than the matched FP32 time for the same bucket size, topology, local fan-in, endpoint service rate, and
network bandwidth"; L275: "losses concentrate under fast networks, high fan-in, and low endpoint service rate".
The paper prints no formula (its times come from replayed NCCL curves), so the time model is reading #20
("parity unpinned by the paper"; pinned by closed forms and by the monotonicities L275 states):
  t_fp32 = 2 (N-1)/N * 4 n / bw                    ring all-reduce of the FP32 bucket over N nodes
  t_hier = F * (p n / 8) / r                       the endpoint counts F local compact updates at r bytes/s (L76)
         + 2 (N-1)/N * (p B n / 8) / bw            partial-count reduction + result return, B = bits of N*F
  admit iff t_hier < t_fp32.       n elements, p planes (1 or 2), F local fan-in, r service rate, bw per-node B/s.
"""
import math

ROUTE_P, ROUTE_L, ROUTE_F = 0, 1, 2
MODE_GBINARY, MODE_GTERNARY = 1, 2


def mgtr(events, bits_binary=1.0, bits_ternary=math.log2(3.0), scale_bytes=4):
    num = den = 0.0
    for numel, route, mode in events:
        fp32 = 4.0 * numel
        den += fp32
        if route == ROUTE_L:
            bits = bits_binary if mode == MODE_GBINARY else bits_ternary
            num += numel * bits / 8.0 + scale_bytes
        else:
            num += fp32
    return num / den if den > 0 else 1.0


def count_planes(w):
    b = 0
    while (1 << b) <= w:
        b += 1
    return b


def guard_times(n, nodes, fan_in, service_rate, bw, planes):
    ring = 2.0 * (nodes - 1) / nodes
    t_fp32 = ring * 4.0 * n / bw
    B = count_planes(nodes * fan_in)
    t_hier = fan_in * (planes * n / 8.0) / service_rate + ring * (planes * B * n / 8.0) / bw
    return t_hier, t_fp32


def guard(n, nodes, fan_in, service_rate, bw, planes):
    t_hier, t_fp32 = guard_times(n, nodes, fan_in, service_rate, bw, planes)
    return 1 if t_hier < t_fp32 else 0
