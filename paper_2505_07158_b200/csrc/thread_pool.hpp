// thread_pool.hpp -- the host worker threads T_w of Algorithm 2, as a fixed pool that runs
// index-parallel jobs (sub-frame hashes, worker-system groups, staging copies).  The paper wakes one thread
// per sub-frame; here the protocol parameter n (how the work is *split*) is independent of how many threads
// *run* it, so results never depend on the machine.
#pragma once
#include <atomic>
#include <condition_variable>
#include <functional>
#include <mutex>
#include <thread>
#include <vector>

namespace vh {

class ThreadPool {
public:
    explicit ThreadPool(unsigned threads) {
        if (threads < 1) threads = 1;
        n_ = threads;
        for (unsigned t = 1; t < threads; ++t) workers_.emplace_back([this] { loop(); });
    }
    ~ThreadPool() {
        {
            std::lock_guard<std::mutex> lk(m_);
            stop_ = true;
            ++epoch_;
        }
        cv_.notify_all();
        for (auto &t : workers_) t.join();
    }
    unsigned size() const { return n_; }

    // Runs fn(i) for i in [0, count) on the pool (the caller takes part); returns when all are done.
    void parallel_for(size_t count, const std::function<void(size_t)> &fn) {
        if (count == 0) return;
        if (n_ == 1 || count == 1) {
            for (size_t i = 0; i < count; ++i) fn(i);
            return;
        }
        {
            std::lock_guard<std::mutex> lk(m_);
            fn_ = &fn;
            count_ = count;
            next_.store(0, std::memory_order_relaxed);
            pending_.store(count, std::memory_order_relaxed);
            ++epoch_;
        }
        cv_.notify_all();
        run();
        std::unique_lock<std::mutex> lk(m_);
        done_cv_.wait(lk, [this] { return pending_.load(std::memory_order_acquire) == 0 && active_ == 0; });
        fn_ = nullptr;
    }

private:
    void run() {
        const std::function<void(size_t)> *fn = fn_;
        const size_t count = count_;
        for (;;) {
            const size_t i = next_.fetch_add(1, std::memory_order_relaxed);
            if (i >= count) break;
            (*fn)(i);
            pending_.fetch_sub(1, std::memory_order_acq_rel);
        }
    }
    void loop() {
        unsigned long seen = 0;
        for (;;) {
            {
                std::unique_lock<std::mutex> lk(m_);
                cv_.wait(lk, [&] { return epoch_ != seen; });
                seen = epoch_;
                if (stop_) return;
                if (!fn_) continue;
                ++active_;
            }
            run();
            {
                std::lock_guard<std::mutex> lk(m_);
                --active_;
            }
            done_cv_.notify_one();
        }
    }

    unsigned n_ = 1;
    std::vector<std::thread> workers_;
    std::mutex m_;
    std::condition_variable cv_, done_cv_;
    unsigned long epoch_ = 0;
    bool stop_ = false;
    const std::function<void(size_t)> *fn_ = nullptr;
    size_t count_ = 0;
    std::atomic<size_t> next_{0}, pending_{0};
    int active_ = 0;
};

}  // namespace vh
