// cd_types.hpp -- host-side construction of token-level automata for typed LM-function outputs
// (section 2.3: return_type / options / quantifier).
// Pure host code (no CUDA): the result is the CSR that cd_compile_dfa takes.
#pragma once
#include <cstdint>
#include <map>
#include <string>
#include <vector>

namespace cdt {

struct HostCsr {
    std::vector<int64_t> row_ptr;
    std::vector<int32_t> tok, next;
    std::vector<uint8_t> accepting;
    int32_t S = 0;
};

struct Builder {
    std::vector<std::map<int, int>> child;  // per state: token -> next state (sorted by token)
    std::vector<uint8_t> acc;
    int add_state() {
        child.emplace_back();
        acc.push_back(0);
        return (int)child.size() - 1;
    }
    // adds (or follows) the transition s --t--> ?, returns the target
    int step(int s, int t) {
        auto it = child[s].find(t);
        if (it != child[s].end()) return it->second;
        const int n = add_state();
        child[s][t] = n;
        return n;
    }
    HostCsr finish() const {
        HostCsr c;
        c.S = (int32_t)child.size();
        c.row_ptr.assign(c.S + 1, 0);
        for (int s = 0; s < c.S; ++s) {
            for (const auto& kv : child[s]) {
                c.tok.push_back(kv.first);
                c.next.push_back(kv.second);
            }
            c.row_ptr[s + 1] = (int64_t)c.tok.size();
        }
        c.accepting = acc;
        return c;
    }
};

// Option set / boolean type (PAPER.md L61 `options`): the trie of K labels (token-id sequences).
//   eos < 0   "a row is finished the first time its state accepts": one accepting leaf per
//             label; labels must be non-empty, distinct and prefix-free (G5: under shortest accept a label
//             that extends another would be unreachable).
//   eos >= 0  the EOS / longest-match variant (G4, G5): language { label + [eos] }.  Every
//             state reached by a whole label ("may stop") gets an eos edge to ONE accepting sink; only the
//             sink accepts.  A label may be a token-prefix of another ("New York" / "New York City"): in
//             the shorter label's end state the model either emits eos or goes on.  Labels must be
//             non-empty, distinct and must not contain eos.
// States are numbered in creation order: 0 = root, trie nodes in insertion order (labels in the given
// order, token by token), the sink (eos >= 0) last.
inline std::string build_trie(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok, int32_t eos,
                              HostCsr* out) {
    if (V < 1 || K < 1) return "V and K must be >= 1";
    if (eos >= V) return "eos outside [0, V)";
    if (label_ptr[0] != 0) return "label_ptr[0] must be 0";
    Builder b;
    b.add_state();
    std::vector<uint8_t> ends(1, 0);  // state reached by a whole label
    std::vector<int> end_order;
    for (int k = 0; k < K; ++k) {
        const int64_t lo = label_ptr[k], hi = label_ptr[k + 1];
        if (hi <= lo) return "label " + std::to_string(k) + " is empty";
        int node = 0;
        for (int64_t j = lo; j < hi; ++j) {
            const int t = label_tok[j];
            if (t < 0 || t >= V) return "label " + std::to_string(k) + ": token outside [0, V)";
            if (eos >= 0 && t == eos) return "label " + std::to_string(k) + " contains eos";
            if (eos < 0 && ends[node]) return "label " + std::to_string(k) + " extends another label (not prefix-free)";
            node = b.step(node, t);
            if ((int)ends.size() < (int)b.child.size()) ends.resize(b.child.size(), 0);
        }
        if (ends[node]) return "label " + std::to_string(k) + " duplicates another label";
        if (eos < 0 && !b.child[node].empty()) return "label " + std::to_string(k) + " is a prefix of another label";
        ends[node] = 1;
        end_order.push_back(node);
    }
    if (eos < 0) {
        for (int e : end_order) b.acc[e] = 1;
    } else {
        const int sink = b.add_state();
        b.acc[sink] = 1;
        for (int e : end_order) b.child[e][eos] = sink;
    }
    *out = b.finish();
    return std::string();
}

// Collection type with a quantifier ("{3} for exactly three, {1,5} for between one and
// five"): the language  open item (sep item)^(c-1) close [eos]  for min_items <= c <= max_items (c = 0:
// open close), every item one of K labels (token-id sequences).  One accepting state, reached by the last
// token of `close` (eos < 0) or by eos after it (eos >= 0), so "first accepting state" is
// the end of the list.  Determinism requirements (returned as an error string otherwise): labels
// non-empty and distinct; close non-empty; sep non-empty when max_items > 1; sep[0] != close[0]; when
// min_items == 0, close[0] is not the first token of a label.  eos < 0: labels prefix-free.  eos >= 0
// (longest match): a label may be a token-prefix of another -- the item ends when sep / close follows,
// so in the shorter label's end state sep[0] and close[0] must not continue a longer label; eos occurs
// in no label and in none of open / sep / close.  States are numbered in creation order: 0 = start.
inline std::string build_list(int32_t V, int32_t K, const int64_t* label_ptr, const int32_t* label_tok,
                              const int32_t* open, int32_t n_open, const int32_t* sep, int32_t n_sep,
                              const int32_t* close, int32_t n_close, int32_t min_items, int32_t max_items, int32_t eos,
                              HostCsr* out) {
    if (V < 1 || K < 1) return "V and K must be >= 1";
    if (eos >= V) return "eos outside [0, V)";
    if (min_items < 0 || max_items < min_items || max_items < 1) return "need 0 <= min_items <= max_items, max_items >= 1";
    if (n_close < 1) return "close must hold at least one token";
    if (max_items > 1 && n_sep < 1) return "sep must hold at least one token when max_items > 1";
    if (n_open < 0 || n_sep < 0) return "negative length";
    auto in_range = [&](const int32_t* p, int n) {
        for (int i = 0; i < n; ++i)
            if (p[i] < 0 || p[i] >= V || (eos >= 0 && p[i] == eos)) return false;
        return true;
    };
    if (!in_range(open, n_open) || !in_range(sep, n_sep) || !in_range(close, n_close)) return "token outside [0, V) (or eos inside open / sep / close)";
    if (n_sep > 0 && sep[0] == close[0]) return "sep and close start with the same token";
    if (label_ptr[0] != 0) return "label_ptr[0] must be 0";
    for (int k = 0; k < K; ++k) {
        if (label_ptr[k + 1] <= label_ptr[k]) return "empty label";
        if (!in_range(label_tok + label_ptr[k], (int)(label_ptr[k + 1] - label_ptr[k]))) return "label token outside [0, V) (or eos inside a label)";
        if (min_items == 0 && label_tok[label_ptr[k]] == close[0]) return "close starts like a label while min_items = 0";
    }
    // inner[k]: label k is a proper token-prefix of another label (its end state is an inner trie node)
    std::vector<uint8_t> inner(K, 0);
    for (int k = 0; k < K; ++k)
        for (int q = 0; q < K; ++q) {
            if (q == k) continue;
            const int64_t lk = label_ptr[k + 1] - label_ptr[k], lq = label_ptr[q + 1] - label_ptr[q];
            if (lk > lq) continue;
            bool pre = true;
            for (int64_t j = 0; j < lk && pre; ++j) pre = label_tok[label_ptr[k] + j] == label_tok[label_ptr[q] + j];
            if (!pre) continue;
            if (lk == lq) return "duplicate label or label that is a prefix of another";
            if (eos < 0) return "a label is a prefix of another label";
            inner[k] = 1;
        }
    Builder b;
    int cur = b.add_state();  // start
    for (int i = 0; i < n_open; ++i) cur = b.step(cur, open[i]);
    const int accept = b.add_state();
    b.acc[accept] = 1;
    // the state the last token of close leads to: the accepting state itself, or the state waiting for eos
    int after_close = accept;
    if (eos >= 0) {
        after_close = b.add_state();
        b.child[after_close][eos] = accept;
    }
    auto add_close = [&](int from) {  // from --close--> after_close
        int s = from;
        for (int i = 0; i + 1 < n_close; ++i) s = b.step(s, close[i]);
        if (b.child[s].count(close[n_close - 1]) && b.child[s][close[n_close - 1]] != after_close) return false;
        b.child[s][close[n_close - 1]] = after_close;
        return true;
    };
    // item roots: root = state in which item number c (0-based) starts
    int root = cur;
    if (min_items == 0 && !add_close(root)) return "close collides with the labels";
    for (int c = 0; c < max_items; ++c) {
        // one copy of the label trie hanging off `root`; every label that is not a prefix of another ends in
        // the shared boundary state, the others end in their own (inner) node
        const int boundary = b.add_state();
        std::vector<int> inner_ends;
        for (int k = 0; k < K; ++k) {
            int s = root;
            const int64_t lo = label_ptr[k], hi = label_ptr[k + 1];
            for (int64_t j = lo; j < hi; ++j) {
                if (s == boundary) return "a label is a prefix of another label";
                const bool last = (j + 1 == hi);
                auto it = b.child[s].find(label_tok[j]);
                if (last && !inner[k]) {
                    if (it != b.child[s].end()) return "duplicate label or label that is a prefix of another";
                    b.child[s][label_tok[j]] = boundary;
                } else {
                    if (it != b.child[s].end() && it->second == boundary) return "a label is a prefix of another label";
                    s = b.step(s, label_tok[j]);
                    if (s == accept || s == after_close) return "labels collide with close";
                    if (last) inner_ends.push_back(s);
                }
            }
        }
        const int count = c + 1;
        if (count >= min_items && !add_close(boundary)) return "close collides with sep";
        if (count < max_items) {
            int s = boundary;
            for (int i = 0; i < n_sep; ++i) s = b.step(s, sep[i]);
            root = s;
        }
        // an inner end state continues like the boundary (sep / close), unless that token continues a label
        for (int e : inner_ends)
            for (const auto& kv : b.child[boundary]) {
                if (b.child[e].count(kv.first)) return "sep / close continues a label that extends another label";
                b.child[e][kv.first] = kv.second;
            }
    }
    *out = b.finish();
    return std::string();
}

}  // namespace cdt
